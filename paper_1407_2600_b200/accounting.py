"""Work accounting for the roofline figures: FP32 operations the force kernels execute per useful
interaction, counted from the kernels' arithmetic (force.cu), FFMA = 2 flop, FADD/FMUL = 1, MUFU.RSQ = 0.
Bookkeeping only — none of the method's arithmetic lives here.
"""


def _levels(p):
    for l in range(p + 2):
        for a in range(l, -1, -1):
            for b in range(l - a, -1, -1):
                yield l, a, b, l - a - b


def m2p_ops(p, pot=True):
    """(ffma, fmul, fadd) per cell-particle interaction of k_m2p at order p."""
    ffma, fmul, fadd = 3, 3 + 1, 3          # R2 chain; rho = r * sinv, q = D0^2; r = x - com
    if pot:
        fmul += 1                           # phi = Mhat_0 * D0
    for l in range(1, p + 2):
        fmul += 1 + 3                       # A, u_x[1], u_y[1], u_z[1]
        fadd += 3 * (l - 1)                 # u_i[k] = u_i[k-1] + u_i[1]
        fmul += (l - 1)                     # w[k]
    for l, a, b, c in _levels(p):
        if l == 0:
            continue
        t1 = (a >= 1) + (b >= 1) + (c >= 1)
        t2 = (a >= 2) + (b >= 2) + (c >= 2)
        fmul += 1
        ffma += t1 - 1 + t2                 # recurrence
        ffma += t1                          # gradient contraction
        if pot and l <= p:
            ffma += 1                       # potential contraction
    fmul += 1                               # sinv^2
    ffma += 3 + (1 if pot else 0)           # fold the cell's sums with 1/s^2, 1/s
    return ffma, fmul, fadd


def m2p_flops(p, pot=True):
    f, m, a = m2p_ops(p, pot)
    return 2 * f + m + a


def p2p_ops(pot=True):
    """(ffma, fmul, fadd) per particle-particle interaction of k_p2p."""
    return 6, 3, 3 + (1 if pot else 0)


def p2p_flops(pot=True):
    f, m, a = p2p_ops(pot)
    return 2 * f + m + a


def fp32_peak_flops(n_sm, sm_clock_mhz):
    """nominal FP32 peak: SMs x 128 lanes x 2 flop (FMA) x clock."""
    return n_sm * 128 * 2 * sm_clock_mhz * 1e6


# algorithmic HBM bytes per particle of the streaming phases
BYTES_PER_PARTICLE = {
    "key": 12 + 8 + 4,
    "sort": 8 * (8 + 12 + 12),          # per pass: histogram read 8 + scatter read 12 + write 12
    "gather": 4 + 12 + 4 + 16,
    "scatter": 32 + 4 + 16,
    "kdk": 3 * 36,
}

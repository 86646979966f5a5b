"""Work accounting for the roofline figures: FP32 operations the force kernels execute per useful
interaction, counted from the kernels' arithmetic (force.cu), FFMA = 2 flop, FADD/FMUL = 1, MUFU.RSQ = 0.
Bookkeeping only — none of the method's arithmetic lives here.
"""


def _fr_has(p, q, m, dip=False):
    return m >= q and 2 * m - q <= p and (dip or not (q == 1 and m == 1))


def _rank(q):
    return [(a, b, q - a - b) for a in range(q, -1, -1) for b in range(q - a, -1, -1)]


def m2p_ops(p, pot=True, dip=False):
    """(ffma, fmul, fadd) per cell-particle interaction of k_m2p at order p (pairing form, m2p.cu).
    dip: rows with a dipole block (periodic runs with background subtraction, kernel MODE 2)."""
    ffma, fmul, fadd = 3 + 3, 1, 0          # R2 chain and rho = x * sinv - com'/s (one FMA each); q = h0^2
    fmul += 3 * (p - 1) if p < 3 else 3 * (p - 2) + 1   # rho_i / k, k = 2..p; for p >= 3 the top block needs q/p, not rho_i/p
    for q in range(p + 1):
        if q >= 2 and not (q == p and p >= 3):
            fmul += len(_rank(q))           # monomials of degree q (degree p is never read: its block uses Euler)
        for m in range(q, p + 1):
            if not _fr_has(p, q, m, dip):
                continue
            qfirst_s = 0 if (m == 1 or 2 * m - p < 0) else 2 * m - p
            qfirst_g = max(1, 2 * m - p)
            eul = q >= 3                        # blocks of degree >= 3: value from the gradient (Euler), m2p.cu
            for jj, j in enumerate(_rank(q)):
                if q > 0 and not eul:       # S_m += B mu_j  (q = 0: plain assignment)
                    if q == qfirst_s and jj == 0:
                        fmul += 1
                    else:
                        ffma += 1
                if m >= 2 and q >= 2:       # G_m,i += B mu_{j - e_i}  (q = 1: plain assignment)
                    for i in range(3):
                        if j[i] >= 1:
                            if (q == qfirst_g or eul) and jj == i:
                                fmul += 1
                            else:
                                ffma += 1
            if eul:
                if qfirst_s == q:
                    fmul += 1; ffma += 2    # S_m = (rho/q) . G
                else:
                    ffma += 3
                if qfirst_g != q:
                    fadd += 3               # merge with the lower blocks' gradient
    ffma += 2 * p - 1                       # Horner in q for Pq = sum S_m q^m and its derivative
    fmul += 1; ffma += 1                    # Pq + 2 q Pq'
    ffma += 3 * (p - 1 if dip else p - 2)   # Horner for the gradient sums G_p .. G_2 (.. G_1 with a dipole block)
    fmul += 3 + (2 if dip else 3)           # u = (q (h0 * -1/s^2)) * tt ; k2 = (q (h0 / s^2)) q  (no last q with a dipole block)
    ffma += 6                               # fold the cell's sums into the tile sums
    if pot:
        fmul += 1; ffma += 1
    return ffma, fmul, fadd


def m2p_flops(p, pot=True, dip=False):
    f, m, a = m2p_ops(p, pot, dip)
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
    "sort": 8 * (8 + 12 + 12),          # N > 2^22: per pass histogram read 8 + scatter read 12 + write 12 (see sort_bytes)
    "gather": 4 + 12 + 4 + 16,
    "scatter": 32 + 4 + 16,
    "kdk": 3 * 36,
}


SORT_ONESWEEP_NMAX = 1 << 22            # DSK_SORT_ONESWEEP_NMAX of csrc/dsk_internal.cuh


def sort_bytes(n):
    """algorithmic HBM bytes per particle of the radix sort: up to 2^22 keys one read for all eight histograms and one read +
    one write of the 12-byte records per pass (200 B, the figure of SURVEY.md 8(d)); above, a histogram read per pass as well"""
    return 8 + 8 * (12 + 12) if n <= SORT_ONESWEEP_NMAX else BYTES_PER_PARTICLE["sort"]

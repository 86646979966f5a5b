"""fp64 CPU ORACLE for the 2HOT tree-force path — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It shares no code with paper_1407_2600_b200 (the CUDA path) and never calls it.

Written from SURVEY.md §8(c) (readings O1..O9 of PAPER.md:57-79).  Thin ctypes layer over the plain C
in this directory; this file holds no arithmetic of the method except the KDK composition `kdk_step`
(O9), which is three lines of the leapfrog around the C force routines.

Pins (tests/test_oracle_*.py, `-m "not gpu"`): keys (corner cases, bit positions, brute-force
interleave), sort (numpy stable argsort, adversarial inputs), tree (invariants + spatial brute force),
moments (M2M == direct P2M, closed forms), b_n/M2P (closed forms, finite differences, convergence
rate), direct sum (two-body, momentum, uniform/Plummer sphere), tree -> direct as theta -> 0, Ewald
(alpha independence, 2.837297/L, 4 pi/3 limit, symmetric zero points), far field (Taylor vs direct,
trace relations, perfect lattice), KDK (time reversal, free drift, Zel'dovich).  Nothing here is
"parity unpinned".
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

NLEAF = 112   # library constants shared with the CUDA path (O3/O5: the paper leaves them free)
NCRIT = 192
WS = 1     # default half-width of the explicit image block (O7: measured; 2 is the other supported value)
WS_MAX = 2
KEY_LEVELS = 21
FAR_ORDER = 8
BG_DEFAULT = True    # background subtraction (reading O4b) in periodic boxes: on by default on both sides (dsk_set_background)

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        _lib = C.CDLL(path)
        _lib.orc_tree_build.restype = C.c_void_p
        _lib.orc_tree_ncell.restype = C.c_int64
        _lib.orc_tree_ngroup.restype = C.c_int64
        _lib.orc_ewald_self.restype = C.c_double
        _lib.orc_farfield_phi.restype = C.c_double
        _lib.orc_get_threads.restype = C.c_int
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _sink(sink):
    if sink is None:
        return None
    return np.ascontiguousarray(sink, dtype=np.int64)


def nparams(p):
    return (p + 1) * (p + 2) * (p + 3) // 6


def midx(a, b, c):
    l, k = a + b + c, b + c
    return l * (l + 1) * (l + 2) // 6 + k * (k + 1) // 2 + c


def mtable(p):
    """exponent triples in the interface order (rank ascending, a descending, b descending)"""
    out = []
    for l in range(p + 1):
        for a in range(l, -1, -1):
            for b in range(l - a, -1, -1):
                out.append((a, b, l - a - b))
    return out


def threads():
    return int(lib().orc_get_threads())


def set_threads(n):
    lib().orc_set_threads(C.c_int(int(n)))


# ---- O1 / O2 -------------------------------------------------------------------------------------
def keys(pos, box=1.0, periodic=False):
    pos = _f32(pos)
    n = pos.shape[0]
    key = np.empty(n, dtype=np.uint64)
    wrapped = np.empty_like(pos)
    err = lib().orc_keys(C.c_int64(n), _p(pos), C.c_float(box), C.c_int(int(periodic)), _p(key), _p(wrapped))
    if err:
        raise ValueError(f"orc_keys error {err}")
    return key, wrapped


def sort(key):
    key = np.ascontiguousarray(key, dtype=np.uint64)
    n = key.shape[0]
    skey = np.empty(n, dtype=np.uint64)
    order = np.empty(n, dtype=np.uint32)
    lib().orc_sort(C.c_int64(n), _p(key), _p(skey), _p(order))
    return skey, order


# ---- O3-O6 ---------------------------------------------------------------------------------------
class OracleTree:
    def __init__(self, pos, mass, box=1.0, periodic=False, nleaf=NLEAF, ncrit=NCRIT):
        self.pos = _f32(pos)
        self.mass = _f32(mass)
        self.n = self.pos.shape[0]
        self.box = float(box)
        self.periodic = bool(periodic)
        err = C.c_int(0)
        self._h = lib().orc_tree_build(C.c_int64(self.n), _p(self.pos), _p(self.mass), C.c_float(box),
                                       C.c_int(int(periodic)), C.c_int(nleaf), C.c_int(ncrit), C.byref(err))
        if not self._h:
            raise ValueError(f"orc_tree_build error {err.value}")
        self._h = C.c_void_p(self._h)
        self.ncell = int(lib().orc_tree_ncell(self._h))
        self.ngroup = int(lib().orc_tree_ngroup(self._h))
        self.p = -1

    def __del__(self):
        if getattr(self, "_h", None):
            try:
                lib().orc_tree_free(self._h)
            except TypeError:          # interpreter shutdown: the module globals are already gone
                pass
            self._h = None

    def sorted(self):
        skey = np.empty(self.n, dtype=np.uint64)
        order = np.empty(self.n, dtype=np.uint32)
        lib().orc_tree_get_sorted(self._h, _p(skey), _p(order))
        return skey, order

    def wrapped_pos(self):
        out = np.empty((self.n, 3), dtype=np.float32)
        lib().orc_tree_get_wrapped(self._h, _p(out))
        return out

    def cells(self):
        nc = self.ncell
        d = dict(hotkey=np.empty(nc, np.uint64), first=np.empty(nc, np.int64), count=np.empty(nc, np.int64),
                 nchild=np.empty(nc, np.int32), child0=np.empty(nc, np.int64), level=np.empty(nc, np.int32))
        lib().orc_tree_get_cells(self._h, _p(d["hotkey"]), _p(d["first"]), _p(d["count"]), _p(d["nchild"]),
                                 _p(d["child0"]), _p(d["level"]))
        return d

    def groups(self):
        ng = self.ngroup
        d = dict(cell=np.empty(ng, np.int64), first=np.empty(ng, np.int64), count=np.empty(ng, np.int64),
                 bbox=np.empty((ng, 6), np.float32))
        lib().orc_tree_get_groups(self._h, _p(d["cell"]), _p(d["first"]), _p(d["count"]), _p(d["bbox"]))
        return d

    def moments(self, p):
        """fill and return (mass[ncell], com[ncell,3], delta[ncell], M[ncell,NP(p)]) — raw moments"""
        lib().orc_moments(self._h, C.c_int(p))
        self.p = p
        nc, npar = self.ncell, nparams(p)
        cm = np.empty(nc); com = np.empty((nc, 3)); dl = np.empty(nc); mom = np.empty((nc, npar))
        lib().orc_tree_get_moments(self._h, _p(cm), _p(com), _p(dl), _p(mom))
        return cm, com, dl, mom

    def moments_m2m(self, p):
        if self.p != p:
            self.moments(p)
        out = np.empty((self.ncell, nparams(p)))
        lib().orc_moments_m2m(self._h, C.c_int(p), _p(out))
        return out

    def set_mac(self, kind="theta", tol=0.0):
        """acceptance rule of the walks that follow: "theta" (opening angle, O5) or "abs" (error bound <= tol per cell, O5b)"""
        lib().orc_tree_set_mac(self._h, C.c_int(0 if kind == "theta" else 1), C.c_double(tol))

    def mac_bound(self, c, d, sub=False):
        f = lib().orc_mac_bound
        f.restype = C.c_double
        return float(f(self._h, C.c_int64(c), C.c_int(int(sub)), C.c_double(d)))

    def moments_bg(self, p):
        """O4b: (l_b, rho_bar, M'[ntop, NP(p)]) — the moments of particles - rho_bar over the cube of every cell of level <= l_b"""
        if self.p != p:
            self.moments(p)
        lb = C.c_int32(0); ntop = C.c_int64(0); rho = C.c_double(0)
        lib().orc_tree_get_moments_bg(self._h, C.byref(lb), C.byref(ntop), C.byref(rho), None)
        out = np.empty((ntop.value, nparams(p)))
        lib().orc_tree_get_moments_bg(self._h, C.byref(lb), C.byref(ntop), C.byref(rho), _p(out))
        return lb.value, rho.value, out

    def accel(self, eps, theta, p, sink=None, ws=WS, want_pot=True, bg=None):
        """Tr over the explicit image block only (the far field is added by tree_force).  bg: background subtraction
        (reading O4b; periodic trees only)."""
        if self.p != p:
            self.moments(p)
        bg = (BG_DEFAULT if bg is None else bg) and self.periodic
        sink = _sink(sink)
        ns = self.n if sink is None else sink.shape[0]
        acc = np.empty((ns, 3)); pot = np.empty(ns) if want_pot else None
        n_p2p = C.c_int64(0); n_m2p = C.c_int64(0)
        err = lib().orc_tree_accel(self._h, C.c_double(eps), C.c_double(theta), C.c_int(ws), C.c_int(int(bg)), C.c_int64(ns),
                                   _p(sink), _p(acc), _p(pot), C.byref(n_p2p), C.byref(n_m2p))
        if err:
            raise RuntimeError(f"orc_tree_accel error {err}")
        return acc, pot, int(n_p2p.value), int(n_m2p.value)

    def list_counts(self, theta, g, ws=WS):
        if self.p < 0:
            self.moments(2)          # the MAC reads the centres of mass (any order fills them)
        a = C.c_int64(0); b = C.c_int64(0); c = C.c_int64(0)
        lib().orc_group_list_counts(self._h, C.c_double(theta), C.c_int(ws), C.c_int64(g), C.byref(a),
                                    C.byref(b), C.byref(c))
        return int(a.value), int(b.value), int(c.value)


    def lists(self, theta, g, ws=WS, bg=False, full=False):
        """the two interaction lists of group g as (m2p_cell, m2p_img, p2p_cell, p2p_img), walk order; full=True adds
        (m2p_sub, left[k, 6], window[6]): which entries carry subtracted moments, the cubes summed one by one and the
        window, both as inclusive index ranges lo xyz, hi xyz in level-l_b cells (reading O4b)"""
        if self.p < 0:
            self.moments(2)
        nm = C.c_int64(0); npp = C.c_int64(0); nl = C.c_int64(0)
        win = np.zeros(6, np.int64)
        f = lib().orc_group_lists
        f(self._h, C.c_double(theta), C.c_int(ws), C.c_int(int(bg)), C.c_int64(g), C.c_int64(0), None, None, None, C.byref(nm),
          None, None, C.byref(npp), None, C.byref(nl), _p(win))
        cap = max(nm.value, npp.value, nl.value, 1)
        mc = np.empty(cap, np.int64); mi = np.empty(cap, np.int32); ms = np.empty(cap, np.int8)
        pc = np.empty(cap, np.int64); pi = np.empty(cap, np.int32); left = np.empty((cap, 6), np.int64)
        f(self._h, C.c_double(theta), C.c_int(ws), C.c_int(int(bg)), C.c_int64(g), C.c_int64(cap), _p(mc), _p(mi), _p(ms),
          C.byref(nm), _p(pc), _p(pi), C.byref(npp), _p(left), C.byref(nl), _p(win))
        out = (mc[:nm.value], mi[:nm.value], pc[:npp.value], pi[:npp.value])
        return out + (ms[:nm.value].astype(bool), left[:nl.value], win) if full else out


def image_shift(img, box, periodic, ws=WS):
    """image id -> shift vector n L (ids run over ix, iy, iz in {-ws..ws}, iz fastest)"""
    if not periodic:
        return np.zeros(3)
    side = 2 * ws + 1
    return box * np.array([img // (side * side) - ws, (img // side) % side - ws, img % side - ws], dtype=np.float64)


def tree_force(pos, mass, box, periodic, eps, theta, p, sink=None, tree=None, ws=WS, bg=None, mac=None):
    """The whole oracle path Tr: tree sum over the image block (+ O7 far field when periodic).
    bg: background subtraction (reading O4b) in a periodic box; mac: ("theta",) or ("abs", tol) sets the tree's acceptance
    rule (it stays set).  Returns acc, pot, n_p2p, n_m2p, tree."""
    if tree is None:
        tree = OracleTree(pos, mass, box, periodic)
    if mac is not None:
        tree.set_mac(*mac)
    bg = (BG_DEFAULT if bg is None else bg) and bool(periodic)
    acc, pot, n_p2p, n_m2p = tree.accel(eps, theta, p, sink, ws, bg=bg)
    if periodic:
        wp = tree.wrapped_pos()
        lam = farfield_local(wp, mass, box, ws, bg=bg)
        fa, fp = farfield_eval(lam, box, wp, sink)
        acc = acc + fa
        pot = pot + fp
    return acc, pot, n_p2p, n_m2p, tree


def bn(pmax, r, eps2):
    r = np.ascontiguousarray(r, dtype=np.float64)
    b = np.empty(nparams(pmax))
    lib().orc_bn(C.c_int(pmax), _p(r), C.c_double(eps2), _p(b))
    return b


def m2p(p, mom, r, eps2):
    mom = np.ascontiguousarray(mom, dtype=np.float64)
    r = np.ascontiguousarray(r, dtype=np.float64)
    acc = np.zeros(3); pot = C.c_double(0.0)
    lib().orc_m2p(C.c_int(p), _p(mom), _p(r), C.c_double(eps2), _p(acc), C.byref(pot))
    return acc, pot.value


# ---- O4b background subtraction -------------------------------------------------------------------------
def cuboid_field(lo, hi, x):
    """I = int d^3y/|y-x| and g = int (y-x)/|y-x|^3 d^3y over the homogeneous unit-density cuboid [lo, hi]"""
    lo = np.ascontiguousarray(lo, dtype=np.float64); hi = np.ascontiguousarray(hi, dtype=np.float64)
    x = np.ascontiguousarray(x, dtype=np.float64)
    I = C.c_double(0.0); g = np.empty(3)
    lib().orc_cuboid_field(_p(lo), _p(hi), _p(x), C.byref(I), _p(g))
    return I.value, g


def cube_moments(s, ctr, z, p):
    ctr = np.ascontiguousarray(ctr, dtype=np.float64); z = np.ascontiguousarray(z, dtype=np.float64)
    out = np.empty(nparams(p))
    lib().orc_cube_moments(C.c_double(s), _p(ctr), _p(z), C.c_int(p), _p(out))
    return out


def bg_level(n):
    return int(lib().orc_bg_level(C.c_int64(n)))


def bg_halfwidth(theta, lb, ws=WS):
    return int(lib().orc_bg_halfwidth(C.c_double(theta), C.c_int(ws), C.c_int(lb)))


# ---- softening law (O6 / O6b) -----------------------------------------------------------------------------
class softening:
    """`with oracle.softening("k1"):` — every pair term inside the block uses Dehnen's K1 kernel with support h = the `eps` argument
    of the calls (direct sums, tree P2P; the tree's far cells become Newtonian and are accepted only beyond h); "plummer" is the default."""
    def __init__(self, kind):
        self.kind = {"plummer": 0, "k1": 1}[kind]

    def __enter__(self):
        self.old = int(lib().orc_get_softening())
        lib().orc_set_softening(C.c_int(self.kind))
        return self

    def __exit__(self, *a):
        lib().orc_set_softening(C.c_int(self.old))


def soft_pair(r2, length):
    """(f, phi) of the current softening law: acc = -m d f, pot = -m phi"""
    f = C.c_double(0); ph = C.c_double(0)
    lib().orc_soft_pair(C.c_double(r2), C.c_double(length), C.byref(f), C.byref(ph))
    return f.value, ph.value


# ---- D ---------------------------------------------------------------------------------------------
def direct_iso(pos, mass, eps, sink=None):
    pos = _f32(pos); mass = _f32(mass); sink = _sink(sink)
    n = pos.shape[0]; ns = n if sink is None else sink.shape[0]
    acc = np.empty((ns, 3)); pot = np.empty(ns)
    lib().orc_direct_iso(C.c_int64(n), _p(pos), _p(mass), C.c_double(eps), C.c_int64(ns), _p(sink), _p(acc), _p(pot))
    return acc, pot


def direct_per(pos, mass, box, eps, sink=None, ws=WS, alpha=None, pairwise=False):
    pos = _f32(pos); mass = _f32(mass); sink = _sink(sink)
    n = pos.shape[0]; ns = n if sink is None else sink.shape[0]
    alpha = 2.0 / box if alpha is None else alpha
    acc = np.empty((ns, 3)); pot = np.empty(ns)
    fn = lib().orc_direct_per_pairwise if pairwise else lib().orc_direct_per
    fn(C.c_int64(n), _p(pos), _p(mass), C.c_double(box), C.c_double(eps), C.c_int(ws), C.c_double(alpha),
       C.c_int64(ns), _p(sink), _p(acc), _p(pot))
    return acc, pot


def ewald_pair(x, L=1.0, alpha=None, nmax=-1, hmax=-1):
    x = np.ascontiguousarray(x, dtype=np.float64)
    alpha = 2.0 / L if alpha is None else alpha
    psi = C.c_double(0.0); a = np.empty(3)
    lib().orc_ewald_pair(_p(x), C.c_double(L), C.c_double(alpha), C.c_int(nmax), C.c_int(hmax), C.byref(psi), _p(a))
    return psi.value, a


def ewald_self(L=1.0, alpha=None):
    alpha = 2.0 / L if alpha is None else alpha
    return float(lib().orc_ewald_self(C.c_double(L), C.c_double(alpha), C.c_int(-1), C.c_int(-1)))


# ---- O7 --------------------------------------------------------------------------------------------
def farfield_T(L=1.0, ws=WS, order=FAR_ORDER):
    T = np.empty(nparams(order))
    lib().orc_farfield_T(C.c_double(L), C.c_int(ws), C.c_int(order), _p(T))
    return T


def farfield_phi(u, L=1.0, ws=WS):
    u = np.ascontiguousarray(u, dtype=np.float64)
    a = np.empty(3)
    phi = lib().orc_farfield_phi(_p(u), C.c_double(L), C.c_int(ws), _p(a))
    return float(phi), a


def farfield_local(pos, mass, L=1.0, ws=WS, order=FAR_ORDER, bg=False):
    pos = _f32(pos); mass = _f32(mass)
    lam = np.empty(nparams(order))
    lib().orc_farfield_local(C.c_int64(pos.shape[0]), _p(pos), _p(mass), C.c_double(L), C.c_int(ws),
                             C.c_int(order), C.c_int(int(bg)), _p(lam))
    return lam


def farfield_eval(lam, L, pos, sink=None, order=FAR_ORDER):
    pos = _f32(pos); sink = _sink(sink)
    ns = pos.shape[0] if sink is None else sink.shape[0]
    acc = np.empty((ns, 3)); pot = np.empty(ns)
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    lib().orc_farfield_eval(_p(lam), C.c_int(order), C.c_double(L), C.c_int64(ns), _p(pos), _p(sink), _p(acc), _p(pot))
    return acc, pot


# ---- O9 --------------------------------------------------------------------------------------------
def kdk_factors(periodic, mtot, box, a, da, cosmology=None):
    """cosmology = (Omega_m, Omega_Lambda) selects the Friedmann factors (O9b); None: Einstein-de Sitter (O9)."""
    k1 = C.c_double(0); d = C.c_double(0); k2 = C.c_double(0)
    if periodic and cosmology is not None:
        f = lib().orc_kdk_factors_friedmann
        f.restype = None
        f(C.c_double(mtot), C.c_double(box), C.c_double(cosmology[0]), C.c_double(cosmology[1]), C.c_double(a),
          C.c_double(da), C.byref(k1), C.byref(d), C.byref(k2))
        return k1.value, d.value, k2.value
    lib().orc_kdk_factors(C.c_int(int(periodic)), C.c_double(mtot), C.c_double(box), C.c_double(a),
                          C.c_double(da), C.byref(k1), C.byref(d), C.byref(k2))
    return k1.value, d.value, k2.value


def kdk_step(pos, vel, mass, box, periodic, eps, theta, p, a, da, acc=None, force=None, cosmology=None):
    """One KDK step (O9).  State is fp32 (positions/velocities are 32-bit floats); the
    arithmetic of each update is fp64 and the result is rounded once to fp32.  `acc` is the cached
    force at `pos` (None: computed first).  `force(pos)` defaults to the oracle tree force Tr.
    Returns pos', vel', acc' (acc' = force at pos', to be passed to the next step)."""
    pos = _f32(pos).copy(); vel = _f32(vel).copy(); mass = _f32(mass)
    if force is None:
        def force(x):
            return tree_force(x, mass, box, periodic, eps, theta, p)[0]
    mtot = float(np.sum(mass.astype(np.float64)))
    k1, d, k2 = kdk_factors(periodic, mtot, box, a, da, cosmology)
    if acc is None:
        acc = force(pos)
    vel = (vel.astype(np.float64) + acc * k1).astype(np.float32)
    pos = (pos.astype(np.float64) + vel.astype(np.float64) * d).astype(np.float32)
    if periodic:
        pos = keys(pos, box, True)[1]          # the fp32 wrap of O1
    acc = force(pos)
    vel = (vel.astype(np.float64) + acc * k2).astype(np.float32)
    return pos, vel, acc


# ---- O9c: hierarchical (block) time steps --------------------------------------------------------------
def _kick_factor(periodic, mtot, box, a1, a2, cosmology=None):
    """K(a1, a2) = int dt/a over [a1, a2] (isolated: a2 - a1), through the O9/O9b factors."""
    return kdk_factors(periodic, mtot, box, a1, 2.0 * (a2 - a1), cosmology)[0]


def _drift_factor(periodic, mtot, box, a1, a2, cosmology=None):
    return kdk_factors(periodic, mtot, box, a1, a2 - a1, cosmology)[1]


def rung_wanted(acc, eps, da, eta, rmax):
    """Rung the step criterion asks for, decided in fp32 (the precision the library decides it in):
    step_i = eta sqrt(eps / |acc_i|), rung = ceil(log2(da / step_i)) clamped to [0, rmax]."""
    a = acc.astype(np.float32)
    amag = np.sqrt(a[:, 0] * a[:, 0] + a[:, 1] * a[:, 1] + a[:, 2] * a[:, 2], dtype=np.float32)
    with np.errstate(divide="ignore", invalid="ignore"):
        step = np.float32(eta) * np.sqrt(np.float32(eps) / amag, dtype=np.float32)
        r = np.ceil(np.log2(np.float32(da) / step, dtype=np.float32))
    r = np.where(np.isfinite(r), r, 0.0)
    return np.clip(r, 0, rmax).astype(np.int64)


def kdk_block_step(pos, vel, mass, rung, box, periodic, eps, theta, p, a, da, rmax, eta, acc=None, cosmology=None):
    """One block step of size da with power-of-two individual steps (reading O9c; "adaptive
    symplectic integrator (Quinn et al. 1997)").  nsub = 2^rmax substeps h = da/nsub; a particle on rung r
    takes steps of L(r) = nsub >> r substeps.  Per substep s: particles whose step starts at s get their
    opening half kick K(a_s, a_s + L h/2); everybody drifts by D(a_s, a_s + h); the particles whose step ends
    at t = s + 1 get new forces (all particles are sources) and their closing half kick K(a_t - L h/2, a_t);
    then their rung follows the criterion: finer at once, coarser by one level and only when t is a multiple
    of the coarser step.  Returns pos', vel', rung', acc' (forces of all particles at a + da)."""
    pos = _f32(pos).copy(); vel = _f32(vel).copy(); mass = _f32(mass)
    rung = np.asarray(rung, dtype=np.int64).copy()
    n = len(pos)
    mtot = float(np.sum(mass.astype(np.float64)))
    nsub = 1 << rmax
    h = da / nsub
    if acc is None:
        acc = tree_force(pos, mass, box, periodic, eps, theta, p)[0]
    acc = np.array(acc, dtype=np.float64)
    for s in range(nsub):
        a_s = a + s * h
        L = nsub >> rung
        start = (s % L) == 0
        K1 = np.array([_kick_factor(periodic, mtot, box, a_s, a_s + (nsub >> r) * h / 2, cosmology) for r in range(rmax + 1)])
        vel[start] = (vel[start].astype(np.float64) + acc[start] * K1[rung[start]][:, None]).astype(np.float32)
        d = _drift_factor(periodic, mtot, box, a_s, a_s + h, cosmology)
        pos = (pos.astype(np.float64) + vel.astype(np.float64) * d).astype(np.float32)
        if periodic:
            pos = keys(pos, box, True)[1]
        t = s + 1
        a_t = a + t * h
        act = (t % L) == 0
        sink = np.nonzero(act)[0]
        acc[sink] = tree_force(pos, mass, box, periodic, eps, theta, p, sink)[0]
        K2 = np.array([_kick_factor(periodic, mtot, box, a_t - (nsub >> r) * h / 2, a_t, cosmology) for r in range(rmax + 1)])
        vel[act] = (vel[act].astype(np.float64) + acc[act] * K2[rung[act]][:, None]).astype(np.float32)
        want = rung_wanted(acc, eps, da, eta, rmax)
        finer = act & (want > rung)
        coarser = act & (want < rung) & (rung > 0) & ((t % (nsub >> np.maximum(rung - 1, 0))) == 0)
        rung[finer] = want[finer]
        rung[coarser] -= 1
    return pos, vel, rung, acc

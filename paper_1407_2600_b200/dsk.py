"""Thin Python binding over the C ABI of libdsk (include/dsk.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the ABI.  PyTorch is used for device memory
(the workspace and the caller's tensors) and streams.  There is no CPU fallback: if libdsk.so is
missing or no CUDA device is present, construction fails loudly.
"""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdsk.so")

SYMBOLS = [
    "dsk_create", "dsk_destroy", "dsk_workspace_bytes", "dsk_bind_workspace", "dsk_set_stream",
    "dsk_set_params", "dsk_build_tree", "dsk_accel", "dsk_accel_active", "dsk_accel_shard", "dsk_kdk_step", "dsk_kdk_block_step", "dsk_kdk_reset", "dsk_set_cosmology", "dsk_set_walk_mode", "dsk_set_walk_sharing", "dsk_get_walk_info", "dsk_set_background", "dsk_get_background", "dsk_set_image_block", "dsk_get_image_block", "dsk_set_mac", "dsk_set_softening", "dsk_get_bg_moments", "dsk_get_keys",
    "dsk_get_tree", "dsk_get_moments", "dsk_get_moments_scaled", "dsk_get_groups", "dsk_get_stats", "dsk_get_param", "dsk_get_task_widths",
    "dsk_get_lattice_tensors", "dsk_probe_fp32_peak", "dsk_probe_fp32_peak_ex", "dsk_sort_keys_noalloc", "dsk_strerror",
]


class DskStats(C.Structure):
    _fields_ = [(k, C.c_int64) for k in ("n", "ncell", "nleaf_cells", "ngroup", "nlevel", "n_p2p", "n_m2p",
                                         "list_m2p", "list_p2p", "nbatch", "n_launch", "list_bg")] + \
               [(k, C.c_float) for k in ("ms_key", "ms_sort", "ms_build", "ms_upward", "ms_group", "ms_walk",
                                         "ms_p2p", "ms_m2p", "ms_far", "ms_scatter", "ms_kdk")]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class DskError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"dsk error {code}: {msg}")
        self.code = code


_lib = None


def load_library(path=LIB_PATH):
    """dlopen libdsk.so and declare the prototypes (no compute call is made)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise ImportError(f"{path} not found: build it with `python -m paper_1407_2600_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(path)
    vp, i64, f32, i32, f64 = C.c_void_p, C.c_int64, C.c_float, C.c_int, C.c_double
    lib.dsk_create.argtypes = [C.POINTER(vp), i64, f32, i32, f32, f32, i32]
    lib.dsk_destroy.argtypes = [vp]
    lib.dsk_workspace_bytes.argtypes = [vp]
    lib.dsk_workspace_bytes.restype = C.c_size_t
    lib.dsk_bind_workspace.argtypes = [vp, vp, C.c_size_t]
    lib.dsk_set_stream.argtypes = [vp, vp]
    lib.dsk_set_params.argtypes = [vp, f32, f32, i32]
    lib.dsk_build_tree.argtypes = [vp, vp, vp]
    lib.dsk_accel.argtypes = [vp, vp, vp, vp, vp]
    lib.dsk_accel_active.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.dsk_accel_shard.argtypes = [vp, i32, i32, vp, vp, C.POINTER(i64), C.POINTER(i64)]
    lib.dsk_kdk_step.argtypes = [vp, vp, vp, vp, f64, f64]
    lib.dsk_kdk_block_step.argtypes = [vp, vp, vp, vp, vp, f64, f64, i32, f32]
    lib.dsk_kdk_reset.argtypes = [vp]
    lib.dsk_set_walk_mode.argtypes = [vp, i32]
    lib.dsk_set_walk_sharing.argtypes = [vp, i32]
    lib.dsk_get_walk_info.argtypes = [vp, C.POINTER(i32), C.POINTER(i64)]
    lib.dsk_set_background.argtypes = [vp, i32]
    lib.dsk_set_mac.argtypes = [vp, i32, f32]
    lib.dsk_set_softening.argtypes = [vp, i32, f32]
    lib.dsk_set_image_block.argtypes = [vp, i32]
    lib.dsk_get_image_block.argtypes = [vp, C.POINTER(i32)]
    lib.dsk_get_background.argtypes = [vp, C.POINTER(i32), C.POINTER(i32), C.POINTER(i32), C.POINTER(i64), C.POINTER(f64)]
    lib.dsk_get_bg_moments.argtypes = [vp, vp]
    lib.dsk_set_cosmology.argtypes = [vp, f64, f64]
    lib.dsk_get_keys.argtypes = [vp, vp, vp]
    lib.dsk_get_tree.argtypes = [vp, C.POINTER(i64), vp, vp, vp, vp]
    lib.dsk_get_moments.argtypes = [vp, vp, vp]
    lib.dsk_get_moments_scaled.argtypes = [vp, vp, vp]
    lib.dsk_get_groups.argtypes = [vp, C.POINTER(i64), vp, vp, vp, vp, vp]
    lib.dsk_get_stats.argtypes = [vp, C.POINTER(DskStats)]
    lib.dsk_get_param.argtypes = [C.c_char_p, C.POINTER(f64)]
    lib.dsk_get_task_widths.argtypes = [C.c_int, C.POINTER(C.c_int)]
    lib.dsk_get_lattice_tensors.argtypes = [vp, vp]
    lib.dsk_probe_fp32_peak.argtypes = [i32, C.POINTER(f64), C.POINTER(f64), C.POINTER(f64)]
    lib.dsk_probe_fp32_peak_ex.argtypes = [i32, C.POINTER(f64), C.POINTER(f64), C.POINTER(f64), C.POINTER(f64)]
    lib.dsk_sort_keys_noalloc.argtypes = [vp, i64, f32, i32, vp, vp, vp]
    lib.dsk_strerror.argtypes = [i32]
    lib.dsk_strerror.restype = C.c_char_p
    for s in SYMBOLS:
        if s not in ("dsk_workspace_bytes", "dsk_strerror"):
            getattr(lib, s).restype = i32
    _lib = lib
    return lib


def get_param(name):
    v = C.c_double(0)
    _check(load_library().dsk_get_param(name.encode(), C.byref(v)))
    return v.value


def get_task_widths(n):
    w = (C.c_int * 4)()
    _check(load_library().dsk_get_task_widths(int(n), w))
    return [int(x) for x in w if x]


def probe_fp32_peak(variant):
    """dsk_probe_fp32_peak: (TFLOP/s, cycles per warp instruction per SM sub-partition, SM MHz) of a pure FMA kernel"""
    t, c, m = C.c_double(0), C.c_double(0), C.c_double(0)
    _check(load_library().dsk_probe_fp32_peak(int(variant), C.byref(t), C.byref(c), C.byref(m)))
    return t.value, c.value, m.value


def probe_fp32_peak_ex(variant):
    """(TFLOP/s by CUDA events, cycles per warp instruction per sub-partition, SM MHz, TFLOP/s by the SMs' cycle counters)"""
    t, c, m, tc = C.c_double(0), C.c_double(0), C.c_double(0), C.c_double(0)
    _check(load_library().dsk_probe_fp32_peak_ex(int(variant), C.byref(t), C.byref(c), C.byref(m), C.byref(tc)))
    return t.value, c.value, m.value, tc.value


def sort_keys_noalloc(pos, box, periodic, sorted_keys, order, stream=None):
    """dsk_sort_keys_noalloc: Morton keys + sort of pos [N, 3] (N <= NOALLOC_NMAX) into the caller's sorted_keys (int64 bit
    pattern of uint64) and order (int32 bit pattern of uint32), both CUDA [N].  Allocates nothing, here or in the library;
    calls that overlap on one GPU race on the library's fixed scratch array."""
    pos = _dev_f32(pos)
    n = pos.shape[0]
    if pos.dim() != 2 or pos.shape[1] != 3:
        raise ValueError("pos must be [N, 3]")
    for t, dt in ((sorted_keys, torch.int64), (order, torch.int32)):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dt and t.is_contiguous() and t.numel() == n
                and t.device == pos.device):
            raise TypeError("sorted_keys / order: contiguous CUDA tensors [N] of int64 / int32 on pos's device")
    with torch.cuda.device(pos.device):
        st = torch.cuda.current_stream().cuda_stream if stream is None else stream
        _check(load_library().dsk_sort_keys_noalloc(_ptr(pos), n, float(box), int(bool(periodic)), _ptr(sorted_keys),
                                                    _ptr(order), C.c_void_p(st)))


NOALLOC_NMAX = 1 << 20      # DSK_NOALLOC_NMAX of include/dsk.h


def _check(code):
    if code != 0:
        raise DskError(code, load_library().dsk_strerror(code).decode())


def nparams(p):
    return (p + 1) * (p + 2) * (p + 3) // 6


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


def _dev_f32(t, shape=None):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError("expected a contiguous float32 CUDA tensor")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"expected shape {shape}, got {tuple(t.shape)}")
    return t


class Dsk:
    """One dsk_ctx plus the torch-owned workspace it borrows."""

    def __init__(self, N, box=1.0, periodic=False, eps=1e-3, theta=0.5, p=4, device="cuda:0", stream=None, p_max=None):
        """p_max: the highest order set_params will be asked for (the workspace is sized for it)."""
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("dsk needs a CUDA device (sm_100a); there is no CPU fallback")
        self.device = torch.device(device)
        self.N, self.box, self.periodic = int(N), float(box), bool(periodic)
        self.eps, self.theta, self.p = float(eps), float(theta), int(p)
        h = C.c_void_p(0)
        p_create = max(self.p, int(p_max)) if p_max is not None else self.p
        _check(self.lib.dsk_create(C.byref(h), self.N, self.box, int(self.periodic), self.eps, self.theta, p_create))
        self._h = h
        if p_create != self.p:
            _check(self.lib.dsk_set_params(self._h, self.eps, self.theta, self.p))
        with torch.cuda.device(self.device):
            nbytes = self.lib.dsk_workspace_bytes(self._h)
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = (self.workspace.data_ptr() + 255) & ~255
            s = stream if stream is not None else torch.cuda.current_stream(self.device)
            _check(self.lib.dsk_set_stream(self._h, C.c_void_p(s.cuda_stream)))
            _check(self.lib.dsk_bind_workspace(self._h, C.c_void_p(base), nbytes))
        self.workspace_bytes = nbytes

    def close(self):
        if getattr(self, "_h", None):
            self.lib.dsk_destroy(self._h)
            self._h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the calls of include/dsk.h ------------------------------------------------------------------
    def set_stream(self, stream):
        _check(self.lib.dsk_set_stream(self._h, C.c_void_p(stream.cuda_stream)))

    def set_params(self, eps=None, theta=None, p=None):
        self.eps = self.eps if eps is None else float(eps)
        self.theta = self.theta if theta is None else float(theta)
        self.p = self.p if p is None else int(p)
        _check(self.lib.dsk_set_params(self._h, self.eps, self.theta, self.p))

    def build_tree(self, pos, mass):
        _dev_f32(pos, (self.N, 3)); _dev_f32(mass, (self.N,))
        _check(self.lib.dsk_build_tree(self._h, _ptr(pos), _ptr(mass)))

    def accel(self, pos, mass, acc=None, pot=None, want_pot=True):
        _dev_f32(pos, (self.N, 3)); _dev_f32(mass, (self.N,))
        if acc is None:
            acc = torch.empty((self.N, 3), dtype=torch.float32, device=self.device)
        if pot is None and want_pot:
            pot = torch.empty(self.N, dtype=torch.float32, device=self.device)
        _check(self.lib.dsk_accel(self._h, _ptr(pos), _ptr(mass), _ptr(_dev_f32(acc, (self.N, 3))),
                                  _ptr(pot) if pot is not None else None))
        return acc, pot

    def accel_active(self, pos, mass, active, acc, pot=None):
        """forces of the particles with active[i] != 0 (uint8 CUDA tensor [N]) written into acc/pot in place"""
        _dev_f32(pos, (self.N, 3)); _dev_f32(mass, (self.N,)); _dev_f32(acc, (self.N, 3))
        if not (active.is_cuda and active.dtype == torch.uint8 and active.is_contiguous() and active.numel() == self.N):
            raise TypeError("active: contiguous uint8 CUDA tensor [N]")
        _check(self.lib.dsk_accel_active(self._h, _ptr(pos), _ptr(mass), C.c_void_p(active.data_ptr()), _ptr(acc),
                                         _ptr(pot) if pot is not None else None))
        return acc, pot

    def accel_shard(self, rank, nranks, acc, pot=None):
        """forces of this rank's work-weighted run of sink groups, written into acc/pot in place; returns the run [first, end)"""
        _dev_f32(acc, (self.N, 3))
        lo, hi = C.c_int64(0), C.c_int64(0)
        _check(self.lib.dsk_accel_shard(self._h, int(rank), int(nranks), _ptr(acc), _ptr(pot) if pot is not None else None,
                                        C.byref(lo), C.byref(hi)))
        return lo.value, hi.value

    def kdk_step(self, pos, vel, mass, a, da):
        _dev_f32(pos, (self.N, 3)); _dev_f32(vel, (self.N, 3)); _dev_f32(mass, (self.N,))
        _check(self.lib.dsk_kdk_step(self._h, _ptr(pos), _ptr(vel), _ptr(mass), float(a), float(da)))

    def kdk_block_step(self, pos, vel, mass, rung, a, da, rmax, eta):
        _dev_f32(pos, (self.N, 3)); _dev_f32(vel, (self.N, 3)); _dev_f32(mass, (self.N,))
        if not (rung.is_cuda and rung.dtype == torch.uint8 and rung.is_contiguous() and rung.numel() == self.N):
            raise TypeError("rung: contiguous uint8 CUDA tensor [N]")
        _check(self.lib.dsk_kdk_block_step(self._h, _ptr(pos), _ptr(vel), _ptr(mass), C.c_void_p(rung.data_ptr()),
                                           float(a), float(da), int(rmax), float(eta)))

    def set_softening(self, kind="plummer", length=None):
        """pair softening law: "plummer" (length = eps) or "k1" (Dehnen's K1 kernel, length = its support h)"""
        self.eps = self.eps if length is None else float(length)
        _check(self.lib.dsk_set_softening(self._h, {"plummer": 0, "k1": 1}[kind], self.eps))

    def set_mac(self, kind="theta", tol=0.0):
        """acceptance rule: "theta" (opening angle) or "abs" (absolute error bound tol per cell interaction)"""
        _check(self.lib.dsk_set_mac(self._h, 0 if kind == "theta" else 1, float(tol)))

    def set_image_block(self, ws):
        _check(self.lib.dsk_set_image_block(self._h, int(ws)))

    def get_image_block(self):
        w = C.c_int(0)
        _check(self.lib.dsk_get_image_block(self._h, C.byref(w)))
        return w.value

    def set_background(self, on):
        """0 off, 1 on, 2 on with the windows' background by the closed form everywhere (diagnostic)"""
        _check(self.lib.dsk_set_background(self._h, 2 if on == 2 else int(bool(on))))

    def get_background(self):
        on, lv, k, nt, rho = C.c_int(0), C.c_int(0), C.c_int(0), C.c_int64(0), C.c_double(0)
        _check(self.lib.dsk_get_background(self._h, C.byref(on), C.byref(lv), C.byref(k), C.byref(nt), C.byref(rho)))
        return dict(on=bool(on.value), level=lv.value, halfwidth=k.value, ntop=nt.value, rhobar=rho.value)

    def get_bg_moments(self):
        nt = self.get_background()["ntop"]
        mom = torch.empty((nt, nparams(self.p)), dtype=torch.float32, device=self.device)
        _check(self.lib.dsk_get_bg_moments(self._h, _ptr(mom)))
        return mom

    def set_walk_mode(self, mode):
        _check(self.lib.dsk_set_walk_mode(self._h, int(mode)))

    def set_walk_sharing(self, groups):
        _check(self.lib.dsk_set_walk_sharing(self._h, int(groups)))

    def get_walk_info(self):
        """(the last evaluation walked once into slots predicted from the previous one, evaluations started over so far)"""
        pr, rt = C.c_int(0), C.c_int64(0)
        _check(self.lib.dsk_get_walk_info(self._h, C.byref(pr), C.byref(rt)))
        return bool(pr.value), rt.value

    def set_cosmology(self, omega_m, omega_lambda):
        _check(self.lib.dsk_set_cosmology(self._h, float(omega_m), float(omega_lambda)))

    def kdk_reset(self):
        _check(self.lib.dsk_kdk_reset(self._h))

    # ---- introspection -----------------------------------------------------------------------------------
    def get_keys(self):
        keys = torch.empty(self.N, dtype=torch.int64, device=self.device)       # bit pattern of uint64
        order = torch.empty(self.N, dtype=torch.int32, device=self.device)      # bit pattern of uint32
        _check(self.lib.dsk_get_keys(self._h, _ptr(keys), _ptr(order)))
        return keys, order

    def get_tree(self):
        n = C.c_int64(0)
        _check(self.lib.dsk_get_tree(self._h, C.byref(n), None, None, None, None))
        nc = n.value
        hot = torch.empty(nc, dtype=torch.int64, device=self.device)
        first = torch.empty(nc, dtype=torch.int32, device=self.device)
        count = torch.empty(nc, dtype=torch.int32, device=self.device)
        nchild = torch.empty(nc, dtype=torch.uint8, device=self.device)
        _check(self.lib.dsk_get_tree(self._h, C.byref(n), _ptr(hot), _ptr(first), _ptr(count), _ptr(nchild)))
        return dict(ncell=nc, hotkey=hot, first=first, count=count, nchild=nchild)

    def get_moments(self, scaled=False):
        """scaled=True: moments in units of the cell side, M_n / s^|n| (dsk_get_moments_scaled)"""
        nc = self.get_stats()["ncell"]
        com_mass = torch.empty((nc, 4), dtype=torch.float32, device=self.device)
        mom = torch.empty((nc, nparams(self.p)), dtype=torch.float32, device=self.device)
        f = self.lib.dsk_get_moments_scaled if scaled else self.lib.dsk_get_moments
        _check(f(self._h, _ptr(com_mass), _ptr(mom)))
        return com_mass, mom

    def get_groups(self):
        n = C.c_int64(0)
        _check(self.lib.dsk_get_groups(self._h, C.byref(n), None, None, None, None, None))
        ng = n.value
        first = torch.empty(ng, dtype=torch.int32, device=self.device)
        count = torch.empty(ng, dtype=torch.int32, device=self.device)
        bbox = torch.empty((ng, 6), dtype=torch.float32, device=self.device)
        m2p = torch.empty(ng, dtype=torch.int32, device=self.device)
        p2p = torch.empty(ng, dtype=torch.int32, device=self.device)
        _check(self.lib.dsk_get_groups(self._h, C.byref(n), _ptr(first), _ptr(count), _ptr(bbox), _ptr(m2p), _ptr(p2p)))
        return dict(ngroup=ng, first=first, count=count, bbox=bbox, m2p_len=m2p, p2p_len=p2p)

    def get_stats(self):
        st = DskStats()
        _check(self.lib.dsk_get_stats(self._h, C.byref(st)))
        return st.asdict()

    def get_lattice_tensors(self):
        import numpy as np
        T = np.empty(165, dtype=np.float64)
        _check(self.lib.dsk_get_lattice_tensors(self._h, T.ctypes.data_as(C.c_void_p)))
        return T

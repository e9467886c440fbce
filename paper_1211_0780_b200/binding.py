"""ctypes binding of the C ABI in include/xy.h -- argument marshalling only.

Every step of the Monte Carlo step runs in the CUDA kernels of libxy_b200.so; this module
allocates device memory and a stream through PyTorch (north_star: "PyTorch used only for device
memory and streams"), converts numpy/torch arguments to plain pointers and raises on error
codes.  There is no CPU fallback: a missing library or a missing GPU raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libxy_b200.so")
_lib = None

XY_OPT_TILE_Y, XY_OPT_TILE_Z, XY_OPT_TRACE, XY_OPT_FUSED_MEASURE, XY_OPT_PROFILE, XY_OPT_GENERIC_KERNEL, XY_OPT_OR_PER_MCS, XY_OPT_CUDA_GRAPH, XY_OPT_RESIDENT, XY_OPT_SLOT_CHUNK = 1, 2, 3, 4, 5, 6, 7, 8, 9, 10
KERNEL_CLASSES = ("metropolis", "overrelax", "measure", "finalize", "pt", "other", "fixup", "resident")
NUM_OBS = 5

# name -> (restype, argtypes); tests/test_abi.py checks this table against include/xy.h
_vp, _i, _u64, _sz = C.c_void_p, C.c_int, C.c_uint64, C.c_size_t
_pd, _pf, _pi = C.POINTER(C.c_double), C.POINTER(C.c_float), C.POINTER(C.c_int)
_pu32, _pu64 = C.POINTER(C.c_uint32), C.POINTER(C.c_uint64)
SIGNATURES = {
    "xy_create": (_vp, [_i, _i, _pd, _u64]),
    "xy_destroy": (None, [_vp]),
    "xy_state_bytes": (_sz, [_i, _i]),
    "xy_workspace_bytes": (_sz, [_i, _i]),
    "xy_attach": (_i, [_vp, _vp, _vp, _vp]),
    "xy_init_random": (_i, [_vp]),
    "xy_init_ordered": (_i, [_vp, C.c_float]),
    "xy_set_state": (_i, [_vp, _vp, _i]),
    "xy_get_state": (_i, [_vp, _vp, _i]),
    "xy_metropolis_sweep": (_i, [_vp]),
    "xy_overrelax_sweep": (_i, [_vp]),
    "xy_measure": (_i, [_vp, _vp]),
    "xy_measure_stiffness": (_i, [_vp, _vp]),
    "xy_pt_exchange": (_i, [_vp]),
    "xy_mcs": (_i, [_vp, _i, _vp]),
    "xy_get_perm": (_i, [_vp, _pi]),
    "xy_set_perm": (_i, [_vp, _pi]),
    "xy_get_beta_of_slot": (_i, [_vp, _pd]),
    "xy_set_betas": (_i, [_vp, _pd]),
    "xy_get_counters": (_i, [_vp, _pu32]),
    "xy_set_counters": (_i, [_vp, _pu32]),
    "xy_get_accept_counts": (_i, [_vp, _pu64, _pu64]),
    "xy_get_exact_path_count": (_i, [_vp, _pu64]),
    "xy_set_option": (_i, [_vp, _i, _i]),
    "xy_get_option": (_i, [_vp, _i, _pi]),
    "xy_get_launch_count": (_i, [_vp, _pu64]),
    "xy_get_resident_plan": (_i, [_vp, _pi]),
    "xy_get_kernel_times": (_i, [_vp, _pd, _pu64]),
    "xy_synchronize": (_i, [_vp]),
    "xy_last_error": (C.c_char_p, []),
    "xy_measure_static": (_i, [_vp, _i, _i, _vp, _vp]),
    "xy_debug_get_trace": (_i, [_vp, _vp]),
    "xy_debug_sincos": (_i, [_vp, _vp, _vp, _sz, _vp]),
    "xy_debug_sincos64": (_i, [_vp, _vp, _vp, _sz, _vp]),
    "xy_debug_atan2": (_i, [_vp, _vp, _vp, _sz, _vp]),
    "xy_debug_philox": (_i, [_vp, C.c_uint32, C.c_uint32, _vp, _sz, _vp]),
}


class XYError(RuntimeError):
    pass


def load_library(path=None):
    """dlopen libxy_b200.so and set the prototypes.  Raises if it has not been built."""
    global _lib
    if _lib is None:
        path = path or LIB_PATH
        if not os.path.exists(path):
            raise XYError(f"{path} is missing: build it with `python -m paper_1211_0780_b200.build` "
                          "(there is no CPU fallback)")
        lib = C.CDLL(path)
        for name, (res, args) in SIGNATURES.items():
            f = getattr(lib, name)
            f.restype, f.argtypes = res, args
        _lib = lib
    return _lib


def _check(rc, what):
    if rc != 0:
        msg = load_library().xy_last_error().decode(errors="replace")
        raise XYError(f"{what} failed ({rc}): {msg}")


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise XYError("no CUDA device: paper_1211_0780_b200 has no CPU fallback")
    return torch


def _np_ptr(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


class XY:
    """One (L, R) system on the current CUDA device.  Methods carry the names of include/xy.h.

    The colour-split state and the workspace are torch uint8 tensors owned by this object; the
    kernels run on `stream` (a torch.cuda.Stream; default: the current stream at construction).
    """

    def __init__(self, L, R, betas, seed, stream=None, device=None):
        torch = _torch()
        lib = load_library()
        b = np.ascontiguousarray(betas, dtype=np.float64)
        if b.shape != (R,):
            raise XYError(f"betas must have shape ({R},)")
        self.L, self.R, self.N = int(L), int(R), int(L) ** 3
        self._h = lib.xy_create(self.L, self.R, _np_ptr(b, C.c_double), C.c_uint64(int(seed)))
        if not self._h:
            raise XYError("xy_create failed: " + lib.xy_last_error().decode(errors="replace"))
        self.device = torch.device(device if device is not None else f"cuda:{torch.cuda.current_device()}")
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.current_stream()
            self._state = torch.empty(lib.xy_state_bytes(self.L, self.R), dtype=torch.uint8, device=self.device)
            self._ws = torch.empty(lib.xy_workspace_bytes(self.L, self.R), dtype=torch.uint8, device=self.device)
            _check(lib.xy_attach(self._h, self._state.data_ptr(), self._ws.data_ptr(), self.stream.cuda_stream),
                   "xy_attach")

    def close(self):
        if getattr(self, "_h", None) and load_library is not None:       # None during interpreter shutdown
            load_library().xy_destroy(self._h)
            self._h = None

    __del__ = close

    # ---- state --------------------------------------------------------------------------
    def init_random(self):
        _check(_lib.xy_init_random(self._h), "xy_init_random")

    def init_ordered(self, theta0=0.0):
        _check(_lib.xy_init_ordered(self._h, C.c_float(theta0)), "xy_init_ordered")

    def set_state(self, natural):
        """natural: numpy [R,L,L,L] fp32 (host) or a CUDA torch tensor of R*N fp32."""
        if isinstance(natural, np.ndarray):
            a = np.ascontiguousarray(natural, dtype=np.float32)
            if a.size != self.R * self.N:
                raise XYError("set_state: wrong size")
            _check(_lib.xy_set_state(self._h, a.ctypes.data, 0), "xy_set_state")
        else:
            t = natural
            if t.dtype != _torch().float32 or t.numel() != self.R * self.N or not t.is_contiguous():
                raise XYError("set_state: need a contiguous fp32 tensor of R*N elements")
            on_device = 1 if t.is_cuda else 0
            _check(_lib.xy_set_state(self._h, t.data_ptr(), on_device), "xy_set_state")

    def get_state(self, out=None):
        """Returns numpy [R,L,L,L] fp32, or fills `out` (a contiguous fp32 torch tensor, CUDA or pinned host)."""
        if out is None:
            a = np.empty((self.R, self.L, self.L, self.L), dtype=np.float32)
            _check(_lib.xy_get_state(self._h, a.ctypes.data, 0), "xy_get_state")
            return a
        if out.numel() != self.R * self.N or not out.is_contiguous():
            raise XYError("get_state: need a contiguous fp32 tensor of R*N elements")
        _check(_lib.xy_get_state(self._h, out.data_ptr(), 1 if out.is_cuda else 0), "xy_get_state")
        return out

    # ---- the Monte Carlo step ---------------------------------------------------------------
    def metropolis_sweep(self):
        _check(_lib.xy_metropolis_sweep(self._h), "xy_metropolis_sweep")

    def overrelax_sweep(self):
        _check(_lib.xy_overrelax_sweep(self._h), "xy_overrelax_sweep")

    def measure_stiffness(self):
        """[R, 6] = Cx, Cy, Cz, Sx, Sy, Sz by rank: cos / sin of the bond angle summed per direction (Eq. 6)."""
        out = np.empty((self.R, 6), dtype=np.float64)
        _check(_lib.xy_measure_stiffness(self._h, out.ctypes.data), "xy_measure_stiffness")
        return out

    def measure(self, to_host=True):
        """[R,5] doubles E, Mx, My, |M|^2, |M|^4 by rank; to_host=False only enqueues the reduction."""
        if not to_host:
            _check(_lib.xy_measure(self._h, None), "xy_measure")
            return None
        out = np.empty((self.R, NUM_OBS), dtype=np.float64)
        _check(_lib.xy_measure(self._h, out.ctypes.data), "xy_measure")
        return out

    def measure_static(self, out=None):
        """[R,5] CUDA fp64 tensor E, Mx, My, |M|^2, |M|^4 by SLOT of this object's spins through xy_measure_static, the
        entry point that allocates nothing inside the library (see measure_static below).  Enqueued on self.stream."""
        return measure_static(self._state, self.L, self.R, out=out, stream=self.stream)

    def pt_exchange(self):
        _check(_lib.xy_pt_exchange(self._h), "xy_pt_exchange")

    def mcs(self, n_mcs=1, series=None):
        """n_mcs Monte Carlo steps without host synchronisation; series: CUDA fp64 tensor [n_mcs,R,5] or None."""
        ptr = None
        if series is not None:
            if (not series.is_cuda or series.dtype != _torch().float64 or not series.is_contiguous()
                    or series.numel() != n_mcs * self.R * NUM_OBS):
                raise XYError("mcs: series must be a contiguous CUDA fp64 tensor of n_mcs*R*5 elements")
            ptr = series.data_ptr()
        _check(_lib.xy_mcs(self._h, int(n_mcs), ptr), "xy_mcs")

    # ---- bookkeeping --------------------------------------------------------------------------
    def get_perm(self):
        p = np.empty(self.R, dtype=np.int32)
        _check(_lib.xy_get_perm(self._h, _np_ptr(p, C.c_int)), "xy_get_perm")
        return p

    def set_perm(self, perm):
        p = np.ascontiguousarray(perm, dtype=np.int32)
        if p.shape != (self.R,):
            raise XYError("set_perm: wrong size")
        _check(_lib.xy_set_perm(self._h, _np_ptr(p, C.c_int)), "xy_set_perm")

    def get_beta_of_slot(self):
        b = np.empty(self.R, dtype=np.float64)
        _check(_lib.xy_get_beta_of_slot(self._h, _np_ptr(b, C.c_double)), "xy_get_beta_of_slot")
        return b

    def set_betas(self, betas):
        b = np.ascontiguousarray(betas, dtype=np.float64)
        if b.shape != (self.R,):
            raise XYError(f"betas must have shape ({self.R},)")
        _check(_lib.xy_set_betas(self._h, _np_ptr(b, C.c_double)), "xy_set_betas")

    def get_counters(self):
        n = np.empty(3, dtype=np.uint32)
        _check(_lib.xy_get_counters(self._h, _np_ptr(n, C.c_uint32)), "xy_get_counters")
        return n

    def set_counters(self, n):
        n = np.ascontiguousarray(n, dtype=np.uint32)
        if n.shape != (3,):
            raise XYError("set_counters: need 3 values")
        _check(_lib.xy_set_counters(self._h, _np_ptr(n, C.c_uint32)), "xy_set_counters")

    def get_accept_counts(self):
        met = np.zeros(self.R, dtype=np.uint64)
        pt = np.zeros(max(self.R - 1, 1), dtype=np.uint64)
        _check(_lib.xy_get_accept_counts(self._h, _np_ptr(met, C.c_uint64), _np_ptr(pt, C.c_uint64)),
               "xy_get_accept_counts")
        return met, pt[: self.R - 1]

    def get_exact_path_count(self):
        n = C.c_uint64(0)
        _check(_lib.xy_get_exact_path_count(self._h, C.byref(n)), "xy_get_exact_path_count")
        return int(n.value)

    def set_option(self, option, value):
        _check(_lib.xy_set_option(self._h, int(option), int(value)), "xy_set_option")

    def get_option(self, option):
        v = C.c_int(0)
        _check(_lib.xy_get_option(self._h, int(option), C.byref(v)), "xy_get_option")
        return int(v.value)

    def get_launch_count(self):
        n = C.c_uint64(0)
        _check(_lib.xy_get_launch_count(self._h, C.byref(n)), "xy_get_launch_count")
        return int(n.value)

    def get_resident_plan(self):
        """{'resident': bool, 'slots_per_block', 'blocks_per_slot', 'threads', 'blocks', 'smem_bytes'} of xy_mcs on this context."""
        out = (C.c_int * 6)()
        _check(_lib.xy_get_resident_plan(self._h, out), "xy_get_resident_plan")
        return dict(zip(("resident", "slots_per_block", "blocks_per_slot", "threads", "blocks", "smem_bytes"), [int(v) for v in out]))

    def get_kernel_times(self):
        """{class: (total ms, launches)} since the last call (needs XY_OPT_PROFILE = 1)."""
        ms = np.zeros(len(KERNEL_CLASSES), dtype=np.float64)
        n = np.zeros(len(KERNEL_CLASSES), dtype=np.uint64)
        _check(_lib.xy_get_kernel_times(self._h, _np_ptr(ms, C.c_double), _np_ptr(n, C.c_uint64)), "xy_get_kernel_times")
        return {k: (float(ms[i]), int(n[i])) for i, k in enumerate(KERNEL_CLASSES)}

    def synchronize(self):
        _check(_lib.xy_synchronize(self._h), "xy_synchronize")

    def debug_get_trace(self):
        a = np.empty((self.R, self.L, self.L, self.L), dtype=np.float32)
        _check(_lib.xy_debug_get_trace(self._h, a.ctypes.data), "xy_debug_get_trace")
        return a


# ---- the reduction for callers that cannot allocate device memory ------------------------------
def measure_static(state, L, R, out=None, stream=None):
    """xy_measure_static of include/xy.h: observables by SLOT of a colour-split state the caller already holds.

    The library allocates nothing in this call -- its scratch is a 1 MiB array compiled into libxy_b200.so -- which is
    the point: it serves code that is lent a spin state but cannot get device memory of its own (everything already
    given to another pool, no cudaMalloc allowed in a loop that must not stall, a fixed memory budget).  Pass `out`
    (contiguous CUDA fp64 tensor of R*5 elements) to keep this wrapper allocation-free too; without it the wrapper
    makes one small torch tensor for convenience.  state: CUDA tensor holding R*L^3 fp32 in the library's colour-split
    layout (XY._state is one).  Asynchronous on `stream` (default: torch's current stream); calls share one scratch
    array per device, so never let two of them overlap on the GPU.  Shapes whose partial sums exceed the array raise."""
    torch = _torch()
    lib = load_library()
    n = int(R) * int(L) ** 3
    if not state.is_cuda or state.numel() * state.element_size() < 4 * n or not state.is_contiguous():
        raise XYError("measure_static: state must be a contiguous CUDA tensor of at least R*L^3 fp32")
    if out is None:
        out = torch.empty((int(R), NUM_OBS), dtype=torch.float64, device=state.device)
    if not out.is_cuda or out.dtype != torch.float64 or not out.is_contiguous() or out.numel() != int(R) * NUM_OBS:
        raise XYError("measure_static: out must be a contiguous CUDA fp64 tensor of R*5 elements")
    with torch.cuda.device(state.device):
        st = stream if stream is not None else torch.cuda.current_stream()
        _check(lib.xy_measure_static(state.data_ptr(), int(L), int(R), out.data_ptr(), st.cuda_stream), "xy_measure_static")
    return out


# ---- test hooks: the kernels' device math on arrays -------------------------------------------
def debug_sincos(x):
    torch = _torch()
    load_library()
    d = torch.as_tensor(np.ascontiguousarray(x, dtype=np.float32)).cuda()
    c, s = torch.empty_like(d), torch.empty_like(d)
    _check(_lib.xy_debug_sincos(d.data_ptr(), c.data_ptr(), s.data_ptr(), d.numel(),
                                torch.cuda.current_stream().cuda_stream), "xy_debug_sincos")
    return c.cpu().numpy(), s.cpu().numpy()


def debug_sincos64(x):
    torch = _torch()
    load_library()
    d = torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64)).cuda()
    c, s = torch.empty_like(d), torch.empty_like(d)
    _check(_lib.xy_debug_sincos64(d.data_ptr(), c.data_ptr(), s.data_ptr(), d.numel(),
                                  torch.cuda.current_stream().cuda_stream), "xy_debug_sincos64")
    return c.cpu().numpy(), s.cpu().numpy()


def debug_atan2(y, x):
    torch = _torch()
    load_library()
    dy = torch.as_tensor(np.ascontiguousarray(y, dtype=np.float32)).cuda()
    dx = torch.as_tensor(np.ascontiguousarray(x, dtype=np.float32)).cuda()
    phi = torch.empty_like(dx)
    _check(_lib.xy_debug_atan2(dy.data_ptr(), dx.data_ptr(), phi.data_ptr(), dx.numel(),
                               torch.cuda.current_stream().cuda_stream), "xy_debug_atan2")
    return phi.cpu().numpy()


def debug_philox(ctr, key0, key1):
    """ctr: [n,4] uint32 -> [n,4] uint32 Philox4x32-10 words from the device implementation."""
    torch = _torch()
    load_library()
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    d = torch.as_tensor(c.view(np.int32)).cuda()
    o = torch.empty_like(d)
    _check(_lib.xy_debug_philox(d.data_ptr(), C.c_uint32(key0), C.c_uint32(key1), o.data_ptr(), c.shape[0],
                                torch.cuda.current_stream().cuda_stream), "xy_debug_philox")
    return o.cpu().numpy().view(np.uint32)

"""Thin Python binding over the C ABI of include/cosenu.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of csrc/.  PyTorch is used for the device workspace
(`torch.empty(..., device='cuda')`) and the stream.  There is NO CPU fallback: if the CUDA library is
missing or no sm_100 device is present, loading / `Cosenu(...)` raises.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libcosenu_b200.so")

FD4_KO3, FV_WENO7 = 0, 1
OK, EINVAL, ENOMEM, ECUDA, ESTATE = 0, 1, 2, 3, 4
OPT_EPS_KO, OPT_WENO_EPS, OPT_ADVECT, OPT_RK_FORM, OPT_STAGE_TIMING, OPT_VARIANT, OPT_QUADRATURE, OPT_KO_ORDER, OPT_GRAPH = 0, 1, 2, 3, 4, 5, 6, 7, 8
OPT_MAX_CTAS = 9
OPT_HALO_TIMEOUT_S = 10

# every symbol include/cosenu.h declares
SYMBOLS = ["cosenu_create", "cosenu_workspace_bytes", "cosenu_attach", "cosenu_set_option", "cosenu_init",
           "cosenu_set_state", "cosenu_step", "cosenu_get_state", "cosenu_get_moments", "cosenu_diagnostics",
           "cosenu_sync", "cosenu_launch_count", "cosenu_stage_times", "cosenu_destroy", "cosenu_last_error",
           "cosenu_create_slab", "cosenu_slab_export", "cosenu_slab_link", "cosenu_slab_push_ghosts",
           "cosenu_slab_ref_sums", "cosenu_slab_set_ref_sums", "cosenu_slab_diag_sums", "cosenu_slab_diag_finish",
           "cosenu_slab_step_group", "cosenu_slab_stage", "cosenu_slab_wait_failed",
           "cosenu_beam_sums_static", "cosenu_beam_sums_static_error", "cosenu_build_id"]
STATIC_MAX_NV = 512   # COSENU_STATIC_MAX_NV of include/cosenu.h


class Diag(C.Structure):
    _fields_ = [("t", C.c_double), ("step", C.c_int64),
                ("psurv_nu", C.c_double), ("psurv_nubar", C.c_double),
                ("dP_max", C.c_double), ("dP_avg", C.c_double),
                ("M0", C.c_double * 3), ("dM0", C.c_double * 3),
                ("trace_dev_max", C.c_double), ("ex_abs_max", C.c_double)]

    def asdict(self):
        return {"t": self.t, "step": self.step, "psurv_nu": self.psurv_nu,
                "psurv_nubar": self.psurv_nubar, "dP_max": self.dP_max, "dP_avg": self.dP_avg,
                "M0": list(self.M0), "dM0": list(self.dM0),
                "trace_dev_max": self.trace_dev_max, "ex_abs_max": self.ex_abs_max}


class SlabPeer(C.Structure):
    """cosenu_slab_peer_t: what a neighbouring slab needs to reach this slab's ghost rows (plain bytes)."""
    _fields_ = [("ipc_handle", C.c_ubyte * 64), ("ipc_offset", C.c_uint64), ("dev_base", C.c_uint64),
                ("pid", C.c_int64), ("device", C.c_int32), ("nvp", C.c_int32), ("nz_local", C.c_int64),
                ("comp_stride", C.c_int64), ("off_buf", C.c_uint64 * 4), ("off_ctr", C.c_uint64)]


_lib = None


def load():
    """Load libcosenu_b200.so (built in-tree by `python -m paper_2203_12866_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("cosenu-b200: %s is missing; run `python -m paper_2203_12866_b200.build` "
                           "(there is no CPU fallback)" % LIB_PATH)
    L = C.CDLL(LIB_PATH)
    dp = C.POINTER(C.c_double)
    L.cosenu_create.restype = C.c_void_p
    L.cosenu_create.argtypes = [C.c_int64, C.c_int32] + [C.c_double] * 5 + [C.c_int]
    L.cosenu_workspace_bytes.restype = C.c_size_t
    L.cosenu_workspace_bytes.argtypes = [C.c_void_p]
    L.cosenu_attach.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
    L.cosenu_set_option.argtypes = [C.c_void_p, C.c_int, C.c_double]
    L.cosenu_init.argtypes = [C.c_void_p, C.c_uint64, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int]
    L.cosenu_set_state.argtypes = [C.c_void_p, C.c_void_p, C.c_double]
    L.cosenu_step.argtypes = [C.c_void_p, C.c_int64]
    L.cosenu_get_state.argtypes = [C.c_void_p, C.c_void_p]
    L.cosenu_get_moments.argtypes = [C.c_void_p, dp]
    L.cosenu_diagnostics.argtypes = [C.c_void_p, C.POINTER(Diag)]
    L.cosenu_sync.argtypes = [C.c_void_p]
    L.cosenu_launch_count.restype = C.c_int64
    L.cosenu_launch_count.argtypes = [C.c_void_p]
    L.cosenu_stage_times.argtypes = [C.c_void_p, dp, C.POINTER(C.c_int64)]
    L.cosenu_destroy.restype = None
    L.cosenu_destroy.argtypes = [C.c_void_p]
    L.cosenu_last_error.restype = C.c_char_p
    L.cosenu_last_error.argtypes = [C.c_void_p]
    L.cosenu_create_slab.restype = C.c_void_p
    L.cosenu_create_slab.argtypes = [C.c_int64, C.c_int64, C.c_int64, C.c_int32] + [C.c_double] * 5 + [C.c_int]
    L.cosenu_slab_export.argtypes = [C.c_void_p, C.POINTER(SlabPeer)]
    L.cosenu_slab_link.argtypes = [C.c_void_p, C.POINTER(SlabPeer), C.POINTER(SlabPeer)]
    L.cosenu_slab_push_ghosts.argtypes = [C.c_void_p]
    L.cosenu_slab_ref_sums.argtypes = [C.c_void_p, dp]
    L.cosenu_slab_set_ref_sums.argtypes = [C.c_void_p, dp]
    L.cosenu_slab_diag_sums.argtypes = [C.c_void_p, dp]
    L.cosenu_slab_diag_finish.argtypes = [C.c_void_p, dp, C.c_int, C.POINTER(Diag)]
    L.cosenu_slab_step_group.argtypes = [C.POINTER(C.c_void_p), C.c_int32, C.c_int64]
    L.cosenu_slab_stage.argtypes = [C.c_void_p, C.c_int32]
    L.cosenu_slab_wait_failed.argtypes = [C.c_void_p, C.POINTER(C.c_int32)]
    L.cosenu_beam_sums_static.argtypes = [C.c_void_p, C.c_int64, C.c_int32, C.c_void_p, C.c_void_p]
    L.cosenu_beam_sums_static_error.restype = C.c_char_p
    L.cosenu_beam_sums_static_error.argtypes = []
    L.cosenu_build_id.restype = C.c_char_p
    L.cosenu_build_id.argtypes = []
    _lib = L
    return L


def build_id():
    """cosenu_build_id: the source hash compiled into the loaded library."""
    return load().cosenu_build_id().decode()


class CosenuError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("cosenu error %d: %s" % (code, msg))
        self.code = code


def beam_sums_static(dev_state, dev_out, stream=None):
    """cosenu_beam_sums_static: per-beam z-sums of |P_nu|, P0_nu, |P_nubar|, P0_nubar of a state that is already on the GPU,
    without any device allocation inside the library (its scratch is an array built into the .so).

    For callers that cannot cudaMalloc where they run: a monitor inside a process whose pooling allocator owns the
    GPU's memory, or one running beside free-running slab handles, where the device-wide wait of cudaFree / cudaMalloc
    would stall a neighbour's halo wait into its time-out.  Both tensors are the caller's: `dev_state` a contiguous CUDA
    float64 tensor (8, nz, nv) with nv <= STATIC_MAX_NV, `dev_out` a contiguous CUDA float64 tensor (4, nv) that is
    overwritten.  This wrapper allocates nothing either; it only passes pointers.  The launches go to `stream` (default:
    torch's current stream) and the call does not wait for them.  All calls on a device share one scratch array: calls
    that may overlap on the GPU must be ordered by the caller.  The first call on a device also looks the array's address
    up; make it outside any stream capture."""
    import torch
    L = load()
    for t in (dev_state, dev_out):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
            raise TypeError("beam_sums_static takes contiguous CUDA float64 tensors")
    if dev_state.dim() != 3 or dev_state.shape[0] != 8 or tuple(dev_out.shape) != (4, dev_state.shape[2]):
        raise ValueError("beam_sums_static: dev_state must be (8, nz, nv) and dev_out (4, nv)")
    st = stream if stream is not None else torch.cuda.current_stream(dev_state.device)
    with torch.cuda.device(dev_state.device):   # the buffers' device must be the current one
        rc = L.cosenu_beam_sums_static(dev_state.data_ptr(), dev_state.shape[1], dev_state.shape[2], dev_out.data_ptr(),
                                       st.cuda_stream)
    if rc != 0:
        raise CosenuError(rc, L.cosenu_beam_sums_static_error().decode())
    return dev_out


class Cosenu:
    """One solver handle on the current CUDA device.  Method names mirror the C ABI."""

    def __init__(self, nz, nv, L, dt, omega, theta, mu, scheme, eps_ko=None, weno_eps=None, advect=True,
                 rk_form=None, variant=0, quadrature=0, ko_order=2, graph=None, use_torch_workspace=True, stream=None, slab=None):
        """slab = (nz_global, z_begin): this handle owns rows [z_begin, z_begin + nz) of a periodic grid of nz_global
        cells (cosenu_create_slab; see slab.py for the drivers)."""
        self._L = load()
        self.nz, self.nv = int(nz), int(nv)
        if slab is None:
            self.h = self._L.cosenu_create(nz, nv, L, dt, omega, theta, mu, scheme)
        else:
            self.h = self._L.cosenu_create_slab(int(slab[0]), int(slab[1]), nz, nv, L, dt, omega, theta, mu, scheme)
        if not self.h:
            raise CosenuError(EINVAL, self._L.cosenu_last_error(None).decode())
        self._ws = None
        if slab is not None and not use_torch_workspace and stream is not None:
            self._chk(self._L.cosenu_attach(self.h, None, 0, stream.cuda_stream))   # library-owned memory, caller's stream
        if use_torch_workspace:
            import torch
            nbytes = self._L.cosenu_workspace_bytes(self.h)
            # torch owns the device memory and the stream; the library only uses them
            self._ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
            st = stream if stream is not None else torch.cuda.current_stream()
            self._chk(self._L.cosenu_attach(self.h, self._ws.data_ptr(), nbytes, st.cuda_stream))
        if eps_ko is not None:
            self.set_option(OPT_EPS_KO, eps_ko)
        if weno_eps is not None:
            self.set_option(OPT_WENO_EPS, weno_eps)
        if not advect:
            self.set_option(OPT_ADVECT, 0)
        if rk_form is not None:
            self.set_option(OPT_RK_FORM, rk_form)
        if variant:
            self.set_option(OPT_VARIANT, variant)
        if quadrature:
            self.set_option(OPT_QUADRATURE, quadrature)
        if ko_order != 2:
            self.set_option(OPT_KO_ORDER, ko_order)
        if graph is not None:
            self.set_option(OPT_GRAPH, 1 if graph else 0)

    def _chk(self, rc):
        if rc != 0:
            raise CosenuError(rc, self._L.cosenu_last_error(self.h).decode())

    def workspace_bytes(self):
        return self._L.cosenu_workspace_bytes(self.h)

    def set_option(self, key, value):
        self._chk(self._L.cosenu_set_option(self.h, key, float(value)))

    def init(self, seed, sigma_nu=0.6, sigma_nubar=0.5, alpha=0.9, pert_amp=1e-6, pert_kind=0):
        self._chk(self._L.cosenu_init(self.h, seed, sigma_nu, sigma_nubar, alpha, pert_amp, pert_kind))

    def set_state(self, state, t=0.0):
        """state: numpy (8, nz, nv) float64, or a host torch tensor (pinned or not) of that shape."""
        if isinstance(state, np.ndarray):
            a = np.ascontiguousarray(state, dtype=np.float64)
            assert a.shape == (8, self.nz, self.nv)
            self._chk(self._L.cosenu_set_state(self.h, a.ctypes.data, t))
        else:
            assert tuple(state.shape) == (8, self.nz, self.nv) and state.is_contiguous() and not state.is_cuda
            self._chk(self._L.cosenu_set_state(self.h, state.data_ptr(), t))

    def step(self, n=1):
        self._chk(self._L.cosenu_step(self.h, n))

    def sync(self):
        self._chk(self._L.cosenu_sync(self.h))

    def get_state(self, out=None):
        if out is None:
            out = np.empty((8, self.nz, self.nv), dtype=np.float64)
        if isinstance(out, np.ndarray):
            assert out.shape == (8, self.nz, self.nv) and out.flags.c_contiguous and out.dtype == np.float64
            self._chk(self._L.cosenu_get_state(self.h, out.ctypes.data))
        else:
            assert tuple(out.shape) == (8, self.nz, self.nv) and out.is_contiguous() and not out.is_cuda
            self._chk(self._L.cosenu_get_state(self.h, out.data_ptr()))
        return out

    def get_moments(self):
        out = np.empty((6, self.nz), dtype=np.float64)
        self._chk(self._L.cosenu_get_moments(self.h, out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    def diagnostics(self):
        d = Diag()
        self._chk(self._L.cosenu_diagnostics(self.h, C.byref(d)))
        return d.asdict()

    def launch_count(self):
        return self._L.cosenu_launch_count(self.h)

    def stage_times(self):
        ms = (C.c_double * 4)()
        n = C.c_int64(0)
        self._chk(self._L.cosenu_stage_times(self.h, ms, C.byref(n)))
        return list(ms), n.value

    def close(self):
        if getattr(self, "h", None):
            self._L.cosenu_destroy(self.h)
            self.h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

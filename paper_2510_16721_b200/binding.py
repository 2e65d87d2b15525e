"""ctypes binding of libcfneb.so -- argument marshalling only; every step of the path runs in the CUDA kernels.

Same names as include/cfneb.h.  PyTorch is used for the device workspace and the stream, nothing else.
There is no CPU fallback: if the library is missing or no CUDA device is present, calls raise.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcfneb.so")

OK, EINVAL, ENOMEM, ECUDA, ENEIGH_OVERFLOW, ECELL, ENAN, ERANGE = 0, -1, -2, -3, -4, -5, -6, -7
POT_LJ_SF, POT_FS_MORSE, POT_SW, POT_DNN, POT_NEP = 0, 1, 2, 3, 4
CELL_FIXED, CELL_B, CELL_D = 0, 1, 2
K_CELLPREP, K_NEIGHBOR, K_FORCE, K_REDUCE, K_SCALAR, K_UPDATE, NKERNELS = 0, 1, 2, 3, 4, 5, 6
KERNEL_CLASSES = ("cell_prep", "neighbor", "force", "reduce", "scalar", "update")

EXPORTS = (
    "cfneb_default_params", "cfneb_workspace_bytes", "cfneb_create", "cfneb_step", "cfneb_step_adaptive", "cfneb_step_timed",
    "cfneb_insert_image", "cfneb_delete_image", "cfneb_adapt", "cfneb_reparametrize", "cfneb_relax_endpoints", "cfneb_get_segment_lengths",
    "cfneb_get_path",
    "cfneb_set_path", "cfneb_get_state", "cfneb_get_checkpoint", "cfneb_set_state", "cfneb_step_hosted", "cfneb_get_forces", "cfneb_get_dots", "cfneb_band_dots_noalloc", "cfneb_band_dots_noalloc_error", "cfneb_get_neighbors", "cfneb_get_status", "cfneb_get_history",
    "cfneb_destroy", "cfneb_strerror", "cfneb_last_cuda_error", "cfneb_util_fp64_peak",
)


class Params(ctypes.Structure):
    """cfneb_params (include/cfneb.h)."""
    _fields_ = [
        ("potential", ctypes.c_int32), ("cell_mode", ctypes.c_int32), ("climb", ctypes.c_int32),
        ("fire_nmin", ctypes.c_int32), ("max_neighbors", ctypes.c_int32), ("max_images", ctypes.c_int32),
        ("rebuild_every", ctypes.c_int32), ("reserved0", ctypes.c_int32),
        ("pot", ctypes.c_double * 12), ("k_spring", ctypes.c_double), ("cell_factor", ctypes.c_double),
        ("fire_dt0", ctypes.c_double), ("fire_dtmax", ctypes.c_double), ("fire_maxstep", ctypes.c_double),
        ("fire_finc", ctypes.c_double), ("fire_fdec", ctypes.c_double), ("fire_astart", ctypes.c_double),
        ("fire_fa", ctypes.c_double), ("skin", ctypes.c_double), ("pressure", ctypes.c_double),
        ("types", ctypes.POINTER(ctypes.c_int32)),
    ]


class Status(ctypes.Structure):
    """cfneb_status (include/cfneb.h)."""
    _fields_ = [
        ("steps", ctypes.c_int64), ("rebuilds", ctypes.c_int64), ("n_images", ctypes.c_int32),
        ("climb_index", ctypes.c_int32), ("error", ctypes.c_int32), ("n_pos", ctypes.c_int32),
        ("max_neighbors_seen", ctypes.c_int32), ("graph_kernel_nodes", ctypes.c_int32), ("fmax", ctypes.c_double),
        ("barrier", ctypes.c_double), ("dt", ctypes.c_double), ("alpha", ctypes.c_double),
        ("cell_factor", ctypes.c_double), ("path_length", ctypes.c_double),
    ]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_ if not k.startswith("reserved")}


class FireState(ctypes.Structure):
    """cfneb_fire_state (include/cfneb.h)."""
    _fields_ = [("dt", ctypes.c_double), ("alpha", ctypes.c_double), ("steps", ctypes.c_int64),
                ("n_pos", ctypes.c_int32), ("first", ctypes.c_int32)]


class HistoryEntry(ctypes.Structure):
    """cfneb_history_entry (include/cfneb.h)."""
    _fields_ = [("step", ctypes.c_int64), ("rebuilds", ctypes.c_int64), ("n_images", ctypes.c_int32),
                ("climb_index", ctypes.c_int32), ("fmax", ctypes.c_double), ("barrier", ctypes.c_double),
                ("dt", ctypes.c_double), ("alpha", ctypes.c_double)]


HISTORY_LEN = 1024  # CFNEB_HISTORY_LEN


class CfnebError(RuntimeError):
    def __init__(self, code, what=""):
        msg = lib().cfneb_strerror(code).decode()
        if code == ECUDA:
            msg += ": " + lib().cfneb_last_cuda_error().decode()
        super().__init__("%s failed: %s (%d)" % (what, msg, code))
        self.code = code


_lib = None


def lib():
    """Load libcfneb.so (built by `python -m paper_2510_16721_b200.build`).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("libcfneb.so not built: run `python -m paper_2510_16721_b200.build` (no CPU fallback exists)")
    L = ctypes.CDLL(LIB_PATH)
    vp, dp, ip = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int32)
    i32, f64 = ctypes.c_int32, ctypes.c_double
    pp = ctypes.POINTER(Params)
    L.cfneb_default_params.restype = None
    L.cfneb_default_params.argtypes = [pp]
    L.cfneb_workspace_bytes.restype = ctypes.c_size_t
    L.cfneb_workspace_bytes.argtypes = [i32, pp]
    L.cfneb_create.restype = ctypes.c_int
    L.cfneb_create.argtypes = [ctypes.POINTER(vp), i32, dp, dp, dp, dp, i32, dp, pp, vp, ctypes.c_size_t, vp]
    for name, args in (
        ("cfneb_step", [vp, i32]), ("cfneb_step_adaptive", [vp, i32, i32, f64, f64]), ("cfneb_step_timed", [vp, i32, dp]), ("cfneb_insert_image", [vp, i32]),
        ("cfneb_delete_image", [vp, i32]), ("cfneb_adapt", [vp, f64, f64, ip, ip]), ("cfneb_reparametrize", [vp, i32]),
        ("cfneb_relax_endpoints", [vp, f64, i32, i32, ip, dp, dp]), ("cfneb_get_segment_lengths", [vp, dp]), ("cfneb_get_path", [vp, ip, dp, dp, dp]),
        ("cfneb_set_path", [vp, dp, dp]), ("cfneb_get_state", [vp, dp, dp]),
        ("cfneb_get_checkpoint", [vp, dp, dp, dp, dp, ctypes.POINTER(FireState)]),
        ("cfneb_set_state", [vp, dp, dp, dp, dp, ctypes.POINTER(FireState)]),
        ("cfneb_step_hosted", [vp, dp, dp, ctypes.POINTER(FireState), i32]),
        ("cfneb_get_forces", [vp, dp, dp, dp, dp]), ("cfneb_get_dots", [vp, dp, dp, dp]), ("cfneb_get_neighbors", [vp, i32, ip, ip, ip]),
        ("cfneb_band_dots_noalloc", [vp, vp, vp, i32, ctypes.c_int64, vp, vp]),
        ("cfneb_get_status", [vp, ctypes.POINTER(Status)]), ("cfneb_util_fp64_peak", [vp, dp]),
        ("cfneb_get_history", [vp, ctypes.c_int64, i32, ctypes.POINTER(HistoryEntry)]),
    ):
        fn = getattr(L, name)
        fn.restype = ctypes.c_int
        fn.argtypes = args
    L.cfneb_destroy.restype = None
    L.cfneb_destroy.argtypes = [vp]
    L.cfneb_strerror.restype = ctypes.c_char_p
    L.cfneb_strerror.argtypes = [ctypes.c_int]
    L.cfneb_last_cuda_error.restype = ctypes.c_char_p
    L.cfneb_last_cuda_error.argtypes = []
    L.cfneb_band_dots_noalloc_error.restype = ctypes.c_char_p
    L.cfneb_band_dots_noalloc_error.argtypes = []
    _lib = L
    return L


def _dptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if a is not None else None


def _iptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)) if a is not None else None


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def default_params(**kw):
    """cfneb_default_params, then overrides.  `pot` may be any sequence of <= 12 numbers; `fire` a dict with the
    keys dt0, dtmax, maxstep, nmin, finc, fdec, astart, fa."""
    p = Params()
    lib().cfneb_default_params(ctypes.byref(p))
    fire = kw.pop("fire", None) or {}
    for k, v in fire.items():
        setattr(p, "fire_" + k, v)
    types = kw.pop("types", None)
    if types is not None:  # kept alive by the Params object: cfneb_create reads it
        p._types = np.ascontiguousarray(types, dtype=np.int32)
        p.types = p._types.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))
    pot = kw.pop("pot", None)
    if pot is not None:
        for k in range(12):
            p.pot[k] = float(pot[k]) if k < len(pot) else 0.0
    for k, v in kw.items():
        if not hasattr(p, k):
            raise KeyError(k)
        setattr(p, k, v)
    return p


def workspace_bytes(n_atoms, params):
    return int(lib().cfneb_workspace_bytes(int(n_atoms), ctypes.byref(params)))


def fp64_peak_tflops():
    import torch
    out = ctypes.c_double(0.0)
    rc = lib().cfneb_util_fp64_peak(ctypes.c_void_p(torch.cuda.current_stream().cuda_stream), ctypes.byref(out))
    if rc:
        raise CfnebError(rc, "cfneb_util_fp64_peak")
    return out.value


NOALLOC_MAX_IMAGES = 128  # CFNEB_NOALLOC_MAX_IMAGES of include/cfneb.h


def band_dots_noalloc(X, G, v, out, stream=None):
    """cfneb_band_dots_noalloc: the ten K4 dot products per image of a band given as CUDA tensors, for code that may not
    allocate device memory: the reduction's scratch is a fixed array inside libcfneb.so, and this wrapper allocates
    nothing either -- `out` is the caller's.  X, G, v: float64, contiguous, [P, ...] with the same number of elements
    per image; out: float64, contiguous, P * 10 elements, same device; at most NOALLOC_MAX_IMAGES images.  Enqueued on
    `stream` (default: torch's current stream on that device) and not waited for.  Calls share one scratch per GPU:
    do not let two of them run concurrently on one device.  The first call on a device does one-time set-up and
    should precede any stream capture."""
    import torch
    P = int(X.shape[0])
    for name, t in (("X", X), ("G", G), ("v", v), ("out", out)):
        if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.device == X.device):
            raise ValueError("%s must be a contiguous float64 CUDA tensor on %s" % (name, X.device))
    if G.shape != X.shape or v.shape != X.shape or out.numel() != P * 10:
        raise ValueError("G and v must have X's shape and out P * 10 elements")
    n_dof = X.numel() // P if P else 0
    with torch.cuda.device(X.device):
        st = stream if stream is not None else torch.cuda.current_stream(X.device)
        rc = lib().cfneb_band_dots_noalloc(ctypes.c_void_p(X.data_ptr()), ctypes.c_void_p(G.data_ptr()), ctypes.c_void_p(v.data_ptr()),
                                           P, n_dof, ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(st.cuda_stream))
    if rc:
        raise CfnebError(rc, "cfneb_band_dots_noalloc: " + lib().cfneb_band_dots_noalloc_error().decode())
    return out


class CFNEB:
    """One band on the GPU.  pos[P,N,3] Cartesian, cells[P,3,3] rows = lattice vectors (or endpoints only with
    n_images).  Methods mirror the C ABI: step, step_timed, insert_image, delete_image, adapt, get_path, ..."""

    def __init__(self, pos, cells, params, n_images=None, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("CFNEB needs a CUDA device (sm_100a); there is no CPU fallback")
        pos, cells = _f64(pos), _f64(cells).reshape(-1, 9)
        self.N = int(pos.shape[1])
        if n_images is None:
            n_images = pos.shape[0]
        explicit = pos.shape[0] == n_images and n_images > 2
        if not explicit and pos.shape[0] != 2:
            raise ValueError("give either all n_images images or the two endpoints")
        self.params = params
        self.device = torch.device(device)
        nbytes = workspace_bytes(self.N, params)
        if nbytes == 0:
            raise CfnebError(EINVAL, "cfneb_workspace_bytes")
        with torch.cuda.device(self.device):
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = (self._ws.data_ptr() + 255) // 256 * 256
            self._stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
            path = None
            if explicit:
                path = np.concatenate([pos[1:-1].reshape(n_images - 2, -1), cells[1:-1]], axis=1)
                path = np.ascontiguousarray(path)
            h = ctypes.c_void_p()
            rc = lib().cfneb_create(ctypes.byref(h), self.N, _dptr(np.ascontiguousarray(pos[0])), _dptr(np.ascontiguousarray(cells[0])),
                                    _dptr(np.ascontiguousarray(pos[-1])), _dptr(np.ascontiguousarray(cells[-1])), int(n_images), _dptr(path),
                                    ctypes.byref(params), ctypes.c_void_p(base), nbytes,
                                    ctypes.c_void_p(self._stream.cuda_stream))
        if rc:
            raise CfnebError(rc, "cfneb_create")
        self._h = h
        self.workspace_bytes = nbytes

    # -- hot path ----------------------------------------------------------------------------------
    def step(self, n=1):
        rc = lib().cfneb_step(self._h, int(n))
        if rc:
            raise CfnebError(rc, "cfneb_step")

    def step_timed(self, n=1):
        ms = np.zeros(NKERNELS)
        rc = lib().cfneb_step_timed(self._h, int(n), _dptr(ms))
        if rc:
            raise CfnebError(rc, "cfneb_step_timed")
        return ms

    def step_adaptive(self, n, adapt_every, d_insert, d_delete):
        """n iterations with the O9 control step taken on the device after every `adapt_every` of them; no
        host synchronisation (cfneb_step_adaptive)."""
        rc = lib().cfneb_step_adaptive(self._h, int(n), int(adapt_every), float(d_insert), float(d_delete))
        if rc:
            raise CfnebError(rc, "cfneb_step_adaptive")

    def synchronize(self):
        self._stream.synchronize()

    @property
    def stream(self):
        return self._stream

    # -- image control -------------------------------------------------------------------------------
    def insert_image(self, after_index):
        rc = lib().cfneb_insert_image(self._h, int(after_index))
        if rc:
            raise CfnebError(rc, "cfneb_insert_image")

    def delete_image(self, index):
        rc = lib().cfneb_delete_image(self._h, int(index))
        if rc:
            raise CfnebError(rc, "cfneb_delete_image")

    def adapt(self, d_insert, d_delete):
        ni, nd = ctypes.c_int32(0), ctypes.c_int32(0)
        rc = lib().cfneb_adapt(self._h, float(d_insert), float(d_delete), ctypes.byref(ni), ctypes.byref(nd))
        if rc:
            raise CfnebError(rc, "cfneb_adapt")
        return ni.value, nd.value

    def reparametrize(self, hold_climbing=True):
        """cfneb_reparametrize: interior images to equal arc length along the band's polyline (asynchronous)."""
        rc = lib().cfneb_reparametrize(self._h, int(bool(hold_climbing)))
        if rc:
            raise CfnebError(rc, "cfneb_reparametrize")

    def relax_endpoints(self, fmax_tol, max_steps, rebuild_band=True):
        """cfneb_relax_endpoints: returns (steps[2], fmax[2], energy[2])."""
        steps = (ctypes.c_int32 * 2)()
        fmax = (ctypes.c_double * 2)()
        en = (ctypes.c_double * 2)()
        rc = lib().cfneb_relax_endpoints(self._h, float(fmax_tol), int(max_steps), int(bool(rebuild_band)), steps, fmax, en)
        if rc:
            raise CfnebError(rc, "cfneb_relax_endpoints")
        return [steps[0], steps[1]], [fmax[0], fmax[1]], [en[0], en[1]]

    # -- views -----------------------------------------------------------------------------------------
    def get_status(self):
        s = Status()
        rc = lib().cfneb_get_status(self._h, ctypes.byref(s))
        if rc:
            raise CfnebError(rc, "cfneb_get_status")
        return s

    def get_history(self, first_step, n):
        """cfneb_get_history: list of n HistoryEntry, the iterations first_step .. first_step + n - 1."""
        out = (HistoryEntry * int(n))()
        rc = lib().cfneb_get_history(self._h, int(first_step), int(n), out)
        if rc:
            raise CfnebError(rc, "cfneb_get_history")
        return list(out)

    @property
    def P(self):
        return int(self.get_status().n_images)

    def get_segment_lengths(self):
        P = self.P
        d = np.zeros(P - 1)
        rc = lib().cfneb_get_segment_lengths(self._h, _dptr(d))
        if rc:
            raise CfnebError(rc, "cfneb_get_segment_lengths")
        return d

    def get_path(self, positions=True):
        P = self.P
        pos = np.zeros((P, self.N, 3)) if positions else None
        cells = np.zeros((P, 3, 3))
        E = np.zeros(P)
        n = ctypes.c_int32(0)
        rc = lib().cfneb_get_path(self._h, ctypes.byref(n), _dptr(pos), _dptr(cells), _dptr(E))
        if rc:
            raise CfnebError(rc, "cfneb_get_path")
        return pos, cells, E

    def get_path_into(self, pos, cells, energies):
        """cfneb_get_path into caller-owned (e.g. pinned) float64 arrays; any may be None."""
        n = ctypes.c_int32(0)
        rc = lib().cfneb_get_path(self._h, ctypes.byref(n), _dptr(pos), _dptr(cells), _dptr(energies))
        if rc:
            raise CfnebError(rc, "cfneb_get_path")
        return n.value

    def set_path(self, pos, cells):
        pos, cells = _f64(pos), _f64(cells)
        rc = lib().cfneb_set_path(self._h, _dptr(pos), _dptr(cells))
        if rc:
            raise CfnebError(rc, "cfneb_set_path")

    def get_state(self):
        P = self.P
        X = np.zeros((P, self.N + 3, 3))
        v = np.zeros((P, self.N + 3, 3))
        rc = lib().cfneb_get_state(self._h, _dptr(X), _dptr(v))
        if rc:
            raise CfnebError(rc, "cfneb_get_state")
        return X, v

    def get_checkpoint(self):
        """cfneb_get_checkpoint: dict(X, v, X_list, list_aux, fire) -- everything cfneb_set_state needs to continue
        the band bit for bit in a new handle."""
        P = self.P
        X, v, Xl = (np.zeros((P, self.N + 3, 3)) for _ in range(3))
        aux = np.zeros((P, 4))
        fire = FireState()
        rc = lib().cfneb_get_checkpoint(self._h, _dptr(X), _dptr(v), _dptr(Xl), _dptr(aux), ctypes.byref(fire))
        if rc:
            raise CfnebError(rc, "cfneb_get_checkpoint")
        return dict(X=X, v=v, X_list=Xl, list_aux=aux, fire=fire)

    def set_state(self, X, v=None, X_list=None, list_aux=None, fire=None):
        """cfneb_set_state; arrays may be caller-owned (e.g. pinned) float64 buffers."""
        X = _f64(X)
        v = _f64(v) if v is not None else None
        X_list = _f64(X_list) if X_list is not None else None
        list_aux = _f64(list_aux) if list_aux is not None else None
        rc = lib().cfneb_set_state(self._h, _dptr(X), _dptr(v), _dptr(X_list), _dptr(list_aux),
                                   ctypes.byref(fire) if fire is not None else None)
        if rc:
            raise CfnebError(rc, "cfneb_set_state")

    def step_hosted(self, X, v=None, fire=None, n_blocks=0):
        """cfneb_step_hosted: one iteration of a band whose state (X, v: C-contiguous float64 arrays, updated in place;
        fire: FireState, updated in place) lives in host memory.  v / fire None: that part stays resident in the handle."""
        for arr in (X, v):
            if arr is not None and not (arr.flags.c_contiguous and arr.dtype == np.float64):
                raise ValueError("X and v must be C-contiguous float64 arrays (they are updated in place)")
        rc = lib().cfneb_step_hosted(self._h, _dptr(X), _dptr(v), ctypes.byref(fire) if fire is not None else None,
                                     int(n_blocks))
        if rc:
            raise CfnebError(rc, "cfneb_step_hosted")

    def get_forces(self, forces=True, f_neb=True):
        P = self.P
        F = np.zeros((P, self.N, 3)) if forces else None
        V = np.zeros((P, 3, 3))
        fn = np.zeros((P, self.N + 3, 3)) if f_neb else None
        E = np.zeros(P)
        rc = lib().cfneb_get_forces(self._h, _dptr(F), _dptr(V), _dptr(fn), _dptr(E))
        if rc:
            raise CfnebError(rc, "cfneb_get_forces")
        return F, V, fn, E

    def get_dots(self, gen_force=True):
        """cfneb_get_dots: (dots[P,10], coef[P,4], G[P,N+3,3]) of a dry evaluation at the current X."""
        P = self.P
        dots, coef = np.zeros((P, 10)), np.zeros((P, 4))
        G = np.zeros((P, self.N + 3, 3)) if gen_force else None
        rc = lib().cfneb_get_dots(self._h, _dptr(dots), _dptr(coef), _dptr(G))
        if rc:
            raise CfnebError(rc, "cfneb_get_dots")
        return dots, coef, G

    def get_neighbors(self, image):
        cap = int(self.params.max_neighbors)
        count = np.zeros(self.N, dtype=np.int32)
        lst = np.zeros((self.N, cap), dtype=np.int32)
        shift = np.zeros((self.N, cap, 3), dtype=np.int32)
        rc = lib().cfneb_get_neighbors(self._h, int(image), _iptr(count), _iptr(lst), _iptr(shift))
        if rc:
            raise CfnebError(rc, "cfneb_get_neighbors")
        return count, lst, shift

    def close(self):
        if getattr(self, "_h", None):
            lib().cfneb_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

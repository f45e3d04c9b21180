"""ctypes binding of libprs (include/prs.h).  Argument marshalling only.

``Simulation`` mirrors the C calls one to one: ``prs_create`` (constructor), ``prs_init``,
``prs_step``, ``prs_diagnostics``, ``prs_copy_out``, ``prs_copy_in``, ``prs_sync``,
``prs_set_option``, ``prs_get_info``, ``prs_destroy``.  The device workspace is a torch uint8 tensor
and the stream is torch's current stream at construction; fields cross the boundary as raw
pointers (torch tensors on the device, or numpy / pinned torch tensors on the host).

There is no CPU fallback: if the library cannot be built or loaded, importing ``lib()`` raises.
"""
import ctypes as C

from . import build as _build

F32, F64 = 0, 1
ARITH_LITERAL, ARITH_COEF, ARITH_FMA = 0, 1, 2
KERNEL_AUTO, KERNEL_GENERIC, KERNEL_TILED, KERNEL_TB2, KERNEL_TBS, KERNEL_CLUSTER, KERNEL_BITS = 0, 1, 2, 3, 4, 5, 6
OPT_STEP_KERNEL, OPT_ARITH, OPT_DIAG_KERNEL, OPT_CHUNK, OPT_TILE_Y, OPT_TB2_TILE_Y, OPT_TBS_STEPS, OPT_TBS_ROWS, OPT_TBS_LOADER, OPT_DIAG_CHUNK, OPT_CLUSTER_CTAS = 1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11
INFO_KERNEL_LAUNCHES, INFO_STEP_KERNEL, INFO_STEP, INFO_DIAG_KERNEL = 1, 2, 3, 4
INFO_HALO_VALID, INFO_HALO_PLANES, INFO_DEVICE = 5, 6, 7
ERR_NAMES = {1: "PRS_ERR_INVALID_ARG", 2: "PRS_ERR_UNSUPPORTED", 3: "PRS_ERR_WORKSPACE",
             4: "PRS_ERR_STATE", 5: "PRS_ERR_CUDA", 6: "PRS_ERR_NOMEM"}

EXPORTS = ["prs_workspace_bytes", "prs_create", "prs_destroy", "prs_init", "prs_step", "prs_diagnostics",
           "prs_weighted_area", "prs_set_beta", "prs_copy_out", "prs_copy_in", "prs_sync", "prs_set_option", "prs_get_info",
           "prs_device_pointers", "prs_last_error", "prs_step_launch_info", "prs_run",
           "prs_diagnostics_static", "prs_diagnostics_static_scratch_bytes", "prs_diagnostics_static_max_sites",
           "prs_slab_workspace_bytes", "prs_create_slab", "prs_slab_halo_regions", "prs_slab_halo_filled", "prs_diag_combine"]


class PrsError(RuntimeError):
    def __init__(self, code, what, detail=""):
        self.code = code
        super().__init__("%s failed: %s%s" % (what, ERR_NAMES.get(code, str(code)), (": " + detail) if detail else ""))


class Diag(C.Structure):
    _fields_ = [("step", C.c_int64), ("eta", C.c_double), ("link_count", C.c_uint64),
                ("wall_sites", C.c_uint64), ("sum_ratio", C.c_double), ("rho", C.c_double),
                ("gv2", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def lib():
    """Loads (building first if the sources changed) paper_1710_10420_b200/libprs.so."""
    global _lib
    if _lib is None:
        # PRS_LIBRARY_VARIANT=jitter loads the race-hunting build (build.py VARIANTS; tests/sanitize_kernels.py)
        import os

        path = _build.build(variant=os.environ.get("PRS_LIBRARY_VARIANT", ""))
        L = C.CDLL(path)
        vp, i64, dbl, u64, ci, sz = C.c_void_p, C.c_int64, C.c_double, C.c_uint64, C.c_int, C.c_size_t
        L.prs_workspace_bytes.argtypes = [ci, i64, ci]
        L.prs_workspace_bytes.restype = sz
        L.prs_create.argtypes = [C.POINTER(vp), ci, i64, ci, dbl, dbl, dbl, dbl, dbl, u64, vp, sz, vp]
        L.prs_destroy.argtypes = [vp]
        L.prs_init.argtypes = [vp, dbl]
        L.prs_step.argtypes = [vp, i64]
        L.prs_diagnostics.argtypes = [vp, C.POINTER(Diag)]
        L.prs_run.argtypes = [vp, i64, i64, C.POINTER(Diag)]
        L.prs_weighted_area.argtypes = [vp, C.POINTER(dbl), C.POINTER(dbl)]
        L.prs_set_beta.argtypes = [vp, dbl]
        L.prs_copy_out.argtypes = [vp, vp, vp]
        L.prs_copy_in.argtypes = [vp, vp, vp, dbl, i64]
        L.prs_sync.argtypes = [vp]
        L.prs_set_option.argtypes = [vp, ci, i64]
        L.prs_get_info.argtypes = [vp, ci, C.POINTER(i64)]
        L.prs_device_pointers.argtypes = [vp, C.POINTER(vp), C.POINTER(vp)]
        L.prs_step_launch_info.argtypes = [vp, C.c_char_p, sz, C.POINTER(i64), C.POINTER(i64), C.POINTER(i64),
                                           C.POINTER(i64), C.POINTER(i64)]
        L.prs_diag_combine.argtypes = [C.POINTER(Diag), ci, ci, i64, C.POINTER(Diag)]
        L.prs_diagnostics_static.argtypes = [ci, i64, ci, dbl, dbl, vp, vp, vp, vp, C.c_char_p, sz]
        L.prs_diagnostics_static_scratch_bytes.argtypes = []
        L.prs_diagnostics_static_scratch_bytes.restype = sz
        L.prs_diagnostics_static_max_sites.argtypes = []
        L.prs_diagnostics_static_max_sites.restype = i64
        L.prs_last_error.argtypes = [vp]
        L.prs_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def prs_workspace_bytes(dims, N, precision):
    return int(lib().prs_workspace_bytes(dims, N, precision))


def diag_combine(parts, dims, N):
    """prs_diag_combine: the lattice's diagnostics from the partial sums of its slabs (dicts of prs_diag fields)."""
    arr = (Diag * len(parts))()
    for a, p in zip(arr, parts):
        for k in ("step", "eta", "link_count", "wall_sites", "sum_ratio"):       # rho, gv2 are outputs
            setattr(a, k, p[k])
    out = Diag()
    rc = lib().prs_diag_combine(arr, len(parts), dims, N, C.byref(out))
    if rc != 0:
        raise PrsError(rc, "prs_diag_combine")
    return out.as_dict()


def diagnostics_static(dims, N, precision, phi, phidot, sums_out, stream=None, W0=10.0, phi0=1.0):
    """prs_diagnostics_static: Eqs. 7-8 on caller-held DEVICE fields with no handle, no workspace and no allocation
    (the scratch is a static device array inside the library; at most 2^27 sites).  phi, phidot: device tensors or
    addresses; sums_out: 24 bytes of device memory (e.g. a torch int64[3] tensor) that receive link_count, wall_sites
    (uint64) and sum_ratio (double); stream: a torch stream or None for the legacy default stream.  Does not synchronise."""
    err = C.create_string_buffer(400)
    rc = lib().prs_diagnostics_static(dims, N, precision, W0, phi0, _raw_pointer(phi), _raw_pointer(phidot),
                                      _raw_pointer(sums_out), None if stream is None else stream.cuda_stream, err, 400)
    if rc != 0:
        raise PrsError(rc, "prs_diagnostics_static", err.value.decode())


def _raw_pointer(obj):
    """Host or device address of a torch tensor / numpy array / int."""
    if obj is None:
        return None
    if isinstance(obj, int):
        return obj
    if hasattr(obj, "data_ptr"):
        return obj.data_ptr()
    if hasattr(obj, "ctypes"):
        return obj.ctypes.data
    raise TypeError("expected a torch tensor, a numpy array or an address")


class Simulation:
    """One PRS simulation on the current CUDA device."""

    def __init__(self, dims, N, precision=F32, alpha=3.0, era_m=1.0, deta=0.1, W0=10.0, phi0=1.0, seed=1,
                 device=None, stream=None):
        import torch  # device memory and streams only

        if not torch.cuda.is_available():
            raise RuntimeError("paper_1710_10420_b200 needs a CUDA device (no CPU fallback)")
        self._torch = torch
        self.dims, self.N, self.precision = int(dims), int(N), int(precision)
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        self.dtype = torch.float32 if precision == F32 else torch.float64
        self.shape = (self.N,) * self.dims
        nbytes = prs_workspace_bytes(dims, N, precision)
        if nbytes == 0:
            raise PrsError(1, "prs_workspace_bytes")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.stream = torch.cuda.current_stream(self.device) if stream is None else stream
            self._h = C.c_void_p()
            rc = lib().prs_create(C.byref(self._h), dims, N, precision, alpha, era_m, deta, W0, phi0, seed,
                                  self.workspace.data_ptr(), nbytes, self.stream.cuda_stream)
        if rc != 0:
            self._h = C.c_void_p()
            raise PrsError(rc, "prs_create")

    # -- plumbing
    def _chk(self, rc, what):
        if rc != 0:
            msg = lib().prs_last_error(self._h)
            raise PrsError(rc, what, msg.decode() if msg else "")

    def close(self):
        if getattr(self, "_h", None):
            lib().prs_destroy(self._h)
            self._h = C.c_void_p()
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C calls
    def init(self, eta0=1.0):
        self._chk(lib().prs_init(self._h, eta0), "prs_init")

    def step(self, nsteps=1):
        self._chk(lib().prs_step(self._h, nsteps), "prs_step")

    def diagnostics(self):
        d = Diag()
        self._chk(lib().prs_diagnostics(self._h, C.byref(d)), "prs_diagnostics")
        return d.as_dict()

    def run(self, ncycles, steps_per_cycle):
        """prs_run: ncycles x (steps_per_cycle steps + diagnostics) in one call; a list of ncycles dicts."""
        arr = (Diag * max(1, ncycles))()
        self._chk(lib().prs_run(self._h, ncycles, steps_per_cycle, arr), "prs_run")
        return [arr[i].as_dict() for i in range(ncycles)]

    def set_beta(self, beta):
        self._chk(lib().prs_set_beta(self._h, beta), "prs_set_beta")

    def weighted_area(self):
        """(area, rho_weighted) of Eq. 7 with the PRS orientation weight."""
        a, r = C.c_double(), C.c_double()
        self._chk(lib().prs_weighted_area(self._h, C.byref(a), C.byref(r)), "prs_weighted_area")
        return float(a.value), float(r.value)

    def copy_out_to(self, phi_dst=None, phidot_dst=None):
        """Copies into caller buffers (torch tensors or numpy arrays, host or device)."""
        self._chk(lib().prs_copy_out(self._h, _raw_pointer(phi_dst), _raw_pointer(phidot_dst)), "prs_copy_out")

    def copy_out(self):
        """Snapshot as two numpy arrays of shape (N,)*dims."""
        import numpy as np

        dt = np.float32 if self.precision == F32 else np.float64
        phi, pd = np.empty(self.shape, dt), np.empty(self.shape, dt)
        self.copy_out_to(phi, pd)
        return phi, pd

    def copy_in(self, phi, phidot, eta0=1.0, step=0):
        import numpy as np

        keep = []
        for a in (phi, phidot):
            if hasattr(a, "data_ptr"):
                if a.dtype != self.dtype or not a.is_contiguous() or a.numel() != self.N ** self.dims:
                    raise ValueError("tensor must be contiguous %s with N^dims elements" % self.dtype)
                keep.append(a)
            else:
                dt = np.float32 if self.precision == F32 else np.float64
                b = np.ascontiguousarray(a, dt)
                if b.size != self.N ** self.dims:
                    raise ValueError("array must have N^dims elements")
                keep.append(b)
        self._chk(lib().prs_copy_in(self._h, _raw_pointer(keep[0]), _raw_pointer(keep[1]), eta0, step), "prs_copy_in")

    def sync(self):
        self._chk(lib().prs_sync(self._h), "prs_sync")

    def set_option(self, option, value):
        self._chk(lib().prs_set_option(self._h, option, value), "prs_set_option")

    def get_info(self, info):
        v = C.c_int64()
        self._chk(lib().prs_get_info(self._h, info, C.byref(v)), "prs_get_info")
        return int(v.value)

    def device_pointers(self):
        p, v = C.c_void_p(), C.c_void_p()
        self._chk(lib().prs_device_pointers(self._h, C.byref(p), C.byref(v)), "prs_device_pointers")
        return p.value, v.value

    def step_launch_info(self):
        """prs_step_launch_info: the main kernel of the last step() call -- name with template arguments, grid,
        block, dynamic shared memory, PRS steps per launch, launches in that call."""
        name = C.create_string_buffer(96)
        grid, block = (C.c_int64 * 3)(), (C.c_int64 * 3)()
        smem, steps, count = C.c_int64(), C.c_int64(), C.c_int64()
        self._chk(lib().prs_step_launch_info(self._h, name, 96, grid, block, C.byref(smem), C.byref(steps),
                                             C.byref(count)), "prs_step_launch_info")
        return {"kernel": name.value.decode(), "grid": [int(v) for v in grid], "block": [int(v) for v in block],
                "smem_bytes": int(smem.value), "steps_per_launch": int(steps.value), "launches": int(count.value)}

    # -- conveniences over set_option / get_info
    def set_step_kernel(self, kernel):
        self.set_option(OPT_STEP_KERNEL, kernel)

    def set_arith(self, arith):
        self.set_option(OPT_ARITH, arith)

    @property
    def kernel_launches(self):
        return self.get_info(INFO_KERNEL_LAUNCHES)

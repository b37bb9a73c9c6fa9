"""Thin Python binding of the C-ABI library (include/ark.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libark_b200.so; PyTorch is used for device
memory (the workspace, the dense state tensors) and the stream.  There is no CPU fallback: if the
library is missing or cannot be loaded this module raises.
"""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# ARK_B200_LIBRARY selects another build of the same C ABI (the strict measuring build of reading A20, kernel tuning
# variants); the default is the in-tree product library
LIB_PATH = os.environ.get("ARK_B200_LIBRARY") or os.path.join(_HERE, "libark_b200.so")

ARK_OK, ARK_EINVAL, ARK_ENOMEM, ARK_ECUDA, ARK_ENONFINITE = 0, -1, -2, -3, -4
BC_PERIODIC, BC_REFLECTING, BC_FIXED_T_WALL, BC_FLUX_WALL = 0, 1, 2, 3

EXPORTS = ["ark_workspace_bytes", "ark_create", "ark_set_state", "ark_get_state", "ark_set_state_host",
           "ark_get_state_host", "ark_compute_dt", "ark_cfl_dt_static", "ark_cfl_dt_static_max_cells", "ark_step", "ark_max_rate_device", "ark_step_device_dt", "ark_run", "ark_set_energy_form", "ark_potential_bytes", "ark_set_potential",
           "ark_halo_bytes", "ark_get_halo", "ark_set_halo", "ark_ke_spectrum_bins", "ark_ke_spectrum",
           "ark_diagnostics", "ark_debug_get_padded",
           "ark_step_kernel_timing", "ark_step_kernel_time", "ark_measure_fp64_peak", "ark_launch_count", "ark_destroy", "ark_last_error", "ark_version_string"]


class ark_bc(C.Structure):
    _fields_ = [("type", (C.c_int * 2) * 3), ("value", (C.c_double * 2) * 3)]


class ArkError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("ark error %d: %s" % (code, msg))
        self.code = code


_lib = None


def load():
    """dlopen libark_b200.so (built in-tree by `python -m paper_1903_09043_b200.build`) and declare prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("%s not found: build it with `python -m paper_1903_09043_b200.build` "
                          "(no CPU fallback exists)" % LIB_PATH)
    lib = C.CDLL(LIB_PATH)
    vp, dp, ip = C.c_void_p, C.c_void_p, C.c_int
    lib.ark_workspace_bytes.argtypes = [ip, ip, ip]
    lib.ark_workspace_bytes.restype = C.c_size_t
    lib.ark_create.argtypes = [C.POINTER(vp), ip, ip, ip, C.c_double, C.c_double, C.POINTER(C.c_double),
                               C.c_double, C.c_double, ip, C.POINTER(ark_bc), vp, C.c_size_t, vp]
    lib.ark_create.restype = ip
    for name in ("ark_set_state", "ark_get_state", "ark_set_state_host", "ark_get_state_host", "ark_debug_get_padded"):
        getattr(lib, name).argtypes = [vp] + [dp] * 5
        getattr(lib, name).restype = ip
    lib.ark_compute_dt.argtypes = [vp, C.c_double, C.POINTER(C.c_double)]
    lib.ark_compute_dt.restype = ip
    lib.ark_cfl_dt_static_max_cells.argtypes = []
    lib.ark_cfl_dt_static_max_cells.restype = C.c_size_t
    lib.ark_cfl_dt_static.argtypes = [ip, ip, ip, C.c_double, C.c_double, C.c_double, C.c_double] + [dp] * 5 + [C.c_double, dp, vp]
    lib.ark_cfl_dt_static.restype = ip
    lib.ark_max_rate_device.argtypes = [vp, dp]
    lib.ark_max_rate_device.restype = ip
    lib.ark_step_device_dt.argtypes = [vp, dp]
    lib.ark_step_device_dt.restype = ip
    lib.ark_step.argtypes = [vp, C.c_double]
    lib.ark_step.restype = ip
    lib.ark_diagnostics.argtypes = [vp, C.POINTER(C.c_double)]
    lib.ark_diagnostics.restype = ip
    lib.ark_run.argtypes = [vp, ip, C.c_double, C.POINTER(C.c_double)]
    lib.ark_run.restype = ip
    lib.ark_set_energy_form.argtypes = [vp, ip]
    lib.ark_set_energy_form.restype = ip
    lib.ark_potential_bytes.argtypes = [ip, ip, ip]
    lib.ark_potential_bytes.restype = C.c_size_t
    lib.ark_set_potential.argtypes = [vp, dp, vp, C.c_size_t]
    lib.ark_set_potential.restype = ip
    lib.ark_ke_spectrum_bins.argtypes = [ip, ip]
    lib.ark_ke_spectrum_bins.restype = ip
    lib.ark_ke_spectrum.argtypes = [vp, C.POINTER(C.c_double), ip]
    lib.ark_ke_spectrum.restype = ip
    lib.ark_halo_bytes.argtypes = [ip, ip, ip]
    lib.ark_halo_bytes.restype = C.c_size_t
    lib.ark_get_halo.argtypes = [vp, ip, dp]
    lib.ark_get_halo.restype = ip
    lib.ark_set_halo.argtypes = [vp, ip, dp]
    lib.ark_set_halo.restype = ip
    lib.ark_step_kernel_timing.argtypes = [vp, ip]
    lib.ark_step_kernel_timing.restype = ip
    lib.ark_step_kernel_time.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_int)]
    lib.ark_step_kernel_time.restype = ip
    lib.ark_measure_fp64_peak.argtypes = [C.POINTER(C.c_double), vp]
    lib.ark_measure_fp64_peak.restype = ip
    lib.ark_launch_count.argtypes = [vp]
    lib.ark_launch_count.restype = C.c_longlong
    lib.ark_destroy.argtypes = [vp]
    lib.ark_destroy.restype = None
    lib.ark_last_error.restype = C.c_char_p
    lib.ark_version_string.restype = C.c_char_p
    _lib = lib
    return lib


def version_string():
    return load().ark_version_string().decode()


def measure_fp64_peak():
    """Sustained fp64 instruction rate of the current device in 1e12 thread-instructions/s (DFMA chains)."""
    out = C.c_double(0.0)
    _check(load().ark_measure_fp64_peak(C.byref(out), C.c_void_p(torch.cuda.current_stream().cuda_stream)))
    return out.value


def workspace_bytes(nx, ny, nz):
    return int(load().ark_workspace_bytes(nx, ny, nz))


def _check(rc):
    if rc != ARK_OK:
        raise ArkError(rc, load().ark_last_error().decode())


def cfl_dt_static_max_cells():
    return int(load().ark_cfl_dt_static_max_cells())


def cfl_dt_static(params, U, cfl, out, stream=None):
    """ark_cfl_dt_static: the CFL time step of a dense device state without a Solver, a workspace or any allocation.

    For callers that have the five fields on the GPU but may not allocate there (a plug-in inside an application whose
    memory pool owns the device, a loop that must avoid the synchronisation of cudaMalloc / cudaFree): the reduction's
    scratch is a fixed array inside the library, so grids are limited to cfl_dt_static_max_cells() = 2^27 cells.
    U: [rho, rhou, rhov, rhow or None (2D), E], contiguous float64 CUDA tensors of nx*ny*nz elements, read in place.
    out: float64 CUDA tensor of 2 elements supplied by the caller; receives [max rate, cfl / max rate].  Asynchronous on
    `stream` (default: torch's current stream); calls that overlap on one GPU race on the shared scratch."""
    lib = load()
    nx, ny, nz = int(params["nx"]), int(params["ny"]), int(params["nz"])
    ptrs = []
    for f, a in enumerate(U):
        if a is None:
            if not (f == 3 and nz == 1):
                raise ValueError("state field %d is None" % f)
            ptrs.append(None)
            continue
        if a.dtype != torch.float64 or not a.is_contiguous() or a.numel() != nx * ny * nz or a.device.type != "cuda":
            raise ValueError("state field %d must be a contiguous float64 CUDA tensor of %d elements" % (f, nx * ny * nz))
        ptrs.append(C.c_void_p(a.data_ptr()))
    if out.dtype != torch.float64 or not out.is_contiguous() or out.numel() != 2 or out.device.type != "cuda":
        raise ValueError("out must be a contiguous float64 CUDA tensor of 2 elements")
    st = stream if stream is not None else torch.cuda.current_stream(out.device)
    _check(lib.ark_cfl_dt_static(nx, ny, nz, float(params["dx"]), float(params["gamma"]), float(params["mu"]),
                                 float(params["kappa"]), *ptrs, float(cfl), C.c_void_p(out.data_ptr()),
                                 C.c_void_p(st.cuda_stream)))
    return out


class _OnDevice:
    """The library's functions, each wrapped so that it runs while `device` is the current CUDA device: a handle belongs
    to the device that was current in ark_create (its kernel attributes, stream and workspace live there), and every entry
    point checks that.  Without this, Solver(device="cuda:1") created while device 0 is current would record device 0."""

    def __init__(self, lib, device):
        index = torch.device(device).index
        self._lib, self._index, self._cache = lib, (torch.cuda.current_device() if index is None else index), {}

    def __getattr__(self, name):
        fn = self._cache.get(name)
        if fn is None:
            raw, index = getattr(self._lib, name), self._index

            def fn(*args):
                with torch.cuda.device(index):
                    return raw(*args)
            self._cache[name] = fn
        return fn


class Solver:
    """ark_create / ark_set_state / ark_get_state / ark_compute_dt / ark_step / ark_run / ark_destroy.

    params: dict(nx, ny, nz, dx, gamma, g, mu, kappa, theta, bc_type[3][2], bc_value[3][2]) as produced by
    `paper_1903_09043_b200.inputs`.  State tensors are dense float64 CUDA tensors of nx*ny*nz elements
    (x fastest); rhow is None in 2D.  Optional keys: energy_form (1 = Appendix B, ark_set_energy_form) and phi (dense
    potential at the cell centres, ark_set_potential).
    """

    def __init__(self, params, device="cuda:0", stream=None):
        lib = load()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1903_09043_b200 needs a CUDA device (no CPU fallback)")
        self.p = dict(params)
        self.device = torch.device(device)
        self.nx, self.ny, self.nz = int(params["nx"]), int(params["ny"]), int(params["nz"])
        self.n = self.nx * self.ny * self.nz
        self.ndim = 3 if self.nz > 1 else 2
        nbytes = lib.ark_workspace_bytes(self.nx, self.ny, self.nz)
        if nbytes == 0:
            raise ArkError(ARK_EINVAL, "invalid grid size")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        base = self.workspace.data_ptr()
        self._ws_ptr = (base + 255) // 256 * 256
        bc = ark_bc()
        for d in range(3):
            for s in range(2):
                bc.type[d][s] = int(params["bc_type"][d][s])
                bc.value[d][s] = float(params["bc_value"][d][s])
        g = (C.c_double * 3)(*[float(x) for x in params["g"]])
        h = C.c_void_p()
        self._lib = _OnDevice(lib, self.device)   # every call below runs with the solver's device current (ark.h)
        _check(self._lib.ark_create(C.byref(h), self.nx, self.ny, self.nz, float(params["dx"]), float(params["gamma"]), g,
                              float(params["mu"]), float(params["kappa"]), int(params["theta"]), C.byref(bc),
                              C.c_void_p(self._ws_ptr), C.c_size_t(nbytes), C.c_void_p(self.stream.cuda_stream)))
        self._h = h
        self._phi_buf = None
        # size queries are answered once here: get_halo / set_halo run every step of a slab run
        self._halo_doubles = int(lib.ark_halo_bytes(self.nx, self.ny, self.nz)) // 8
        self._potential_bytes = int(lib.ark_potential_bytes(self.nx, self.ny, self.nz))
        if int(params.get("energy_form", 0)) != 0:
            self.set_energy_form(int(params["energy_form"]))
        if params.get("phi") is not None:
            self.set_potential(torch.as_tensor(params["phi"], dtype=torch.float64).reshape(-1).to(self.device))

    # ------------------------------------------------------------------ general path (Appendix B, array-valued potential)
    def set_energy_form(self, form):
        _check(self._lib.ark_set_energy_form(self._h, int(form)))

    def set_potential(self, phi):
        """phi: dense float64 CUDA tensor of nx*ny*nz elements (potential at the cell centres), or None for constant g."""
        if phi is None:
            _check(self._lib.ark_set_potential(self._h, None, None, 0))
            self._phi_buf = None
            return
        if phi.dtype != torch.float64 or not phi.is_contiguous() or phi.numel() != self.n or phi.device.type != "cuda":
            raise ValueError("phi must be a contiguous float64 CUDA tensor of %d elements" % self.n)
        nbytes = self._potential_bytes
        buf = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        ptr = (buf.data_ptr() + 255) // 256 * 256
        _check(self._lib.ark_set_potential(self._h, C.c_void_p(phi.data_ptr()), C.c_void_p(ptr), C.c_size_t(nbytes)))
        self._phi_buf = buf                      # the library keeps using it (caller-owned): keep it alive

    # ------------------------------------------------------------------ state
    def _ptrs(self, U, host=False):
        out = []
        for f, a in enumerate(U):
            if a is None:
                if not (f == 3 and self.ndim == 2):
                    raise ValueError("state field %d is None" % f)
                out.append(None)
                continue
            if a.dtype != torch.float64 or not a.is_contiguous() or a.numel() != self.n:
                raise ValueError("state field %d must be a contiguous float64 tensor of %d elements" % (f, self.n))
            if host != (a.device.type == "cpu"):
                raise ValueError("state field %d is on %s" % (f, a.device))
            out.append(C.c_void_p(a.data_ptr()))
        return out

    def set_state(self, U):
        _check(self._lib.ark_set_state(self._h, *self._ptrs(U)))

    def get_state(self, out=None):
        if out is None:
            out = [torch.empty(self.n, dtype=torch.float64, device=self.device) if not (f == 3 and self.ndim == 2) else None
                   for f in range(5)]
        _check(self._lib.ark_get_state(self._h, *self._ptrs(out)))
        return out

    def set_state_host(self, U):
        _check(self._lib.ark_set_state_host(self._h, *self._ptrs(U, host=True)))

    def get_state_host(self, out):
        _check(self._lib.ark_get_state_host(self._h, *self._ptrs(out, host=True)))
        return out

    def get_padded(self):
        """ghost-filled padded state: list of tensors shaped (nz+4 or 1, ny+4, nx+4) (test hook)."""
        shp = ((self.nz + 4) if self.ndim == 3 else 1, self.ny + 4, self.nx + 4)
        out = [torch.empty(shp, dtype=torch.float64, device=self.device) if not (f == 3 and self.ndim == 2) else None
               for f in range(5)]
        ptrs = [None if a is None else C.c_void_p(a.data_ptr()) for a in out]
        _check(self._lib.ark_debug_get_padded(self._h, *ptrs))
        return out

    # ------------------------------------------------------------------ slab decomposition (ARK_BC_EXTERNAL sides)
    def halo_doubles(self):
        return self._halo_doubles

    def get_halo(self, side, out=None):
        """the two interior planes next to z side `side` (0 low, 1 high) with their x / y ghost cells -> CUDA tensor."""
        if out is None:
            out = torch.empty(self.halo_doubles(), dtype=torch.float64, device=self.device)
        _check(self._lib.ark_get_halo(self._h, int(side), C.c_void_p(out.data_ptr())))
        return out

    def set_halo(self, side, buf):
        if buf.dtype != torch.float64 or not buf.is_contiguous() or buf.numel() != self.halo_doubles() or buf.device.type != "cuda":
            raise ValueError("halo must be a contiguous float64 CUDA tensor of %d elements" % self.halo_doubles())
        _check(self._lib.ark_set_halo(self._h, int(side), C.c_void_p(buf.data_ptr())))

    # ------------------------------------------------------------------ time stepping
    def compute_dt(self, cfl):
        dt = C.c_double()
        _check(self._lib.ark_compute_dt(self._h, float(cfl), C.byref(dt)))
        return dt.value

    def step(self, dt):
        _check(self._lib.ark_step(self._h, float(dt)))

    def _one_double(self, t, what):
        if t.dtype != torch.float64 or t.numel() != 1 or t.device != self.workspace.device:
            raise ValueError("%s must be a float64 CUDA tensor of 1 element on %s" % (what, self.workspace.device))
        return C.c_void_p(t.data_ptr())

    def max_rate_device(self, out):
        """ark_max_rate_device: the maximum CFL rate of the current state -> out (1-element CUDA tensor), no host sync."""
        _check(self._lib.ark_max_rate_device(self._h, self._one_double(out, "out")))
        return out

    def step_device_dt(self, dt):
        """ark_step_device_dt: one step whose size is read from the 1-element CUDA tensor dt when the kernels run."""
        _check(self._lib.ark_step_device_dt(self._h, self._one_double(dt, "dt")))

    def run(self, nsteps, cfl, want_dts=False):
        if want_dts:
            buf = (C.c_double * max(nsteps, 1))()
            _check(self._lib.ark_run(self._h, int(nsteps), float(cfl), buf))
            return list(buf)[:nsteps]
        _check(self._lib.ark_run(self._h, int(nsteps), float(cfl), None))
        return None

    def diagnostics(self):
        """-> dict(max_speed, mean_speed, kinetic_energy, max_mach, mass, total_energy) of the current state."""
        buf = (C.c_double * 6)()
        _check(self._lib.ark_diagnostics(self._h, buf))
        return dict(zip(("max_speed", "mean_speed", "kinetic_energy", "max_mach", "mass", "total_energy"), list(buf)))

    def ke_spectrum(self):
        """kinetic-energy power spectrum of the horizontal middle plane -> list over shells kappa."""
        nb = int(self._lib.ark_ke_spectrum_bins(self.nx, self.ny))
        buf = (C.c_double * nb)()
        _check(self._lib.ark_ke_spectrum(self._h, buf, nb))
        return list(buf)

    def step_kernel_timing(self, enable=True):
        _check(self._lib.ark_step_kernel_timing(self._h, int(bool(enable))))

    def step_kernel_time(self):
        """-> (total milliseconds, launches) of the fused step kernel since timing was enabled."""
        ms, n = C.c_double(), C.c_int()
        _check(self._lib.ark_step_kernel_time(self._h, C.byref(ms), C.byref(n)))
        return ms.value, n.value

    def launch_count(self):
        return int(self._lib.ark_launch_count(self._h))

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.ark_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

"""Thin ctypes binding of include/dg_b200.h: argument marshalling only.

PyTorch is used for what the boundary leaves to the caller: device memory (one uint8 workspace
tensor) and the CUDA stream.  Every step of the method runs in the library's CUDA kernels; there
is no fallback of any kind: if libdg_b200.so is missing or a call fails, this raises.
"""
import ctypes
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
_DP = ctypes.POINTER(ctypes.c_double)
_LIB = None

# every symbol include/dg_b200.h declares (tests check the header against this and the .so)
SYMBOLS = {
    "dg_create": (ctypes.c_int, [ctypes.POINTER(ctypes.c_void_p), ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                 ctypes.c_int, ctypes.c_double, _DP]),
    "dg_set_brick": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int]),
    "dg_set_boundary": (ctypes.c_int, [ctypes.c_void_p, ctypes.POINTER(ctypes.c_int), _DP]),
    "dg_variant_count": (ctypes.c_int, [ctypes.c_int]),
    "dg_set_variant": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int]),
    "dg_state_len": (ctypes.c_size_t, [ctypes.c_void_p]),
    "dg_workspace_bytes": (ctypes.c_size_t, [ctypes.c_void_p]),
    "dg_bind": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p]),
    "dg_set_state": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]),
    "dg_residual": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]),
    "dg_max_wavespeed": (ctypes.c_int, [ctypes.c_void_p, _DP]),
    "dg_max_wavespeed_noalloc": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_size_t, ctypes.c_double, ctypes.c_void_p,
                                                ctypes.c_void_p, ctypes.c_char_p, ctypes.c_size_t]),
    "dg_rk_step": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_double, ctypes.c_int]),
    "dg_rk_stage": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_double, ctypes.c_int]),
    "dg_set_spacing": (ctypes.c_int, [ctypes.c_void_p, _DP]),
    "dg_halo_len": (ctypes.c_size_t, [ctypes.c_void_p, ctypes.c_int]),
    "dg_halo_export": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p]),
    "dg_set_halo": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p]),
    "dg_set_halo_pair": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]),
    "dg_set_halo_push": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]),
    "dg_cfl_dt": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_double, ctypes.c_double, _DP]),
    "dg_rk_step_cfl": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_double, ctypes.c_int, _DP, _DP]),
    "dg_get_state": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]),
    "dg_split_volume": (ctypes.c_int, [ctypes.c_void_p]),
    "dg_split_surface": (ctypes.c_int, [ctypes.c_void_p]),
    "dg_split_update": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_double, ctypes.c_int]),
    "dg_split_get_r": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]),
    "dg_set_viscosity": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_double, ctypes.c_double]),
    "dg_split_viscous": (ctypes.c_int, [ctypes.c_void_p]),
    "dg_rk_step_ns": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_double, ctypes.c_int]),
    "dg_nodes": (ctypes.c_int, [ctypes.c_void_p, _DP, _DP]),
    "dg_launch_count": (ctypes.c_ulonglong, [ctypes.c_void_p]),
    "dg_kernel_info": (ctypes.c_int, [ctypes.c_void_p, ctypes.POINTER(ctypes.c_longlong)]),
    "dg_selftest_fastmath": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t,
                                            ctypes.c_void_p]),
    "dg_fp64_peak": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_void_p,
                                    ctypes.POINTER(ctypes.c_ulonglong)]),
    "dg_destroy": (ctypes.c_int, [ctypes.c_void_p]),
    "dg_last_error": (ctypes.c_char_p, [ctypes.c_void_p]),
}
ERRORS = {1: "DG_EINVAL", 2: "DG_EUNSUPPORTED", 3: "DG_ENOMEM", 4: "DG_ECUDA", 5: "DG_ESTATE", 6: "DG_ENONPHYSICAL"}


def selftest_fastmath(x):
    """(1/x, sqrt(x)) of a float64 CUDA tensor as the kernels compute them (dg_selftest_fastmath)."""
    import torch
    lib = load_library()
    assert x.is_cuda and x.dtype == torch.float64 and x.is_contiguous()
    r, q = torch.empty_like(x), torch.empty_like(x)
    rc = lib.dg_selftest_fastmath(x.data_ptr(), r.data_ptr(), q.data_ptr(), x.numel(),
                                  torch.cuda.current_stream(x.device).cuda_stream)
    if rc != 0:
        raise DGError(rc, "dg_selftest_fastmath")
    return r, q


def fp64_peak(device="cuda:0", iters=2048, repeats=5):
    """Measured FP64 FMA rate of the device (thread-level FMA/s) from the library's microbenchmark kernel
    (dg_fp64_peak), timed with CUDA events on the current stream; best of `repeats`."""
    import torch
    lib = load_library()
    dev = torch.device(device)
    with torch.cuda.device(dev):
        sms = torch.cuda.get_device_properties(dev).multi_processor_count
        blocks = sms * 8
        out = torch.empty(blocks * 256, dtype=torch.float64, device=dev)
        stream = torch.cuda.current_stream(dev)
        count = ctypes.c_ulonglong(0)
        best = 0.0
        for _ in range(repeats + 1):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            rc = lib.dg_fp64_peak(out.data_ptr(), blocks, iters, stream.cuda_stream, ctypes.byref(count))
            e1.record(stream)
            if rc != 0:
                raise DGError(rc, "dg_fp64_peak")
            torch.cuda.synchronize(dev)
            best = max(best, count.value / (e0.elapsed_time(e1) * 1e-3))
    return best


NOALLOC_MAX_NODES = 1 << 29      # DG_NOALLOC_MAX_NODES of include/dg_b200.h


def max_wavespeed_noalloc(q, gamma, lam_out, stream=None):
    """dg_max_wavespeed_noalloc: the max wavespeed of a canonical-layout state for callers that cannot give the
    library any device memory (no DG object, no workspace; the library's scratch is a fixed array inside it, so
    at most NOALLOC_MAX_NODES nodes).  `q` is a contiguous float64 CUDA tensor of 5 * n_nodes elements, `lam_out` a
    float64 CUDA tensor of one element on the same device, BOTH provided by the caller -- this function creates no
    tensor either.  The result lands in `lam_out` in the order of `stream` (default: torch's current stream of that
    device); nothing synchronises.  All calls on a device share the library's one scratch array: do not let two of
    them overlap on the GPU.  Returns `lam_out`."""
    import torch
    lib = load_library()
    if not (isinstance(q, torch.Tensor) and q.is_cuda and q.dtype == torch.float64 and q.is_contiguous()):
        raise ValueError("q must be a contiguous float64 CUDA tensor")
    if not (isinstance(lam_out, torch.Tensor) and lam_out.device == q.device and lam_out.dtype == torch.float64
            and lam_out.numel() == 1):
        raise ValueError("lam_out must be a one-element float64 tensor on q's device")
    if q.numel() % 5:
        raise ValueError("q must hold 5 values per node")
    err = ctypes.create_string_buffer(512)
    with torch.cuda.device(q.device):
        s = stream if stream is not None else torch.cuda.current_stream(q.device)
        rc = lib.dg_max_wavespeed_noalloc(q.data_ptr(), q.numel() // 5, float(gamma), lam_out.data_ptr(), s.cuda_stream,
                                          err, len(err))
    if rc != 0:
        raise DGError(rc, err.value.decode())
    return lam_out


class DGError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"{ERRORS.get(code, code)}: {text}")
        self.code = code


def lib_path():
    return os.path.join(HERE, "libdg_b200.so")


def load_library(build_if_missing=True):
    """dlopen libdg_b200.so (building it in-tree with nvcc if it is not there). No fallback."""
    global _LIB
    if _LIB is None:
        path = lib_path()
        if not os.path.exists(path):
            if not build_if_missing:
                raise FileNotFoundError(path)
            from . import build
            build.build()
        lib = ctypes.CDLL(path)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(lib, name)      # AttributeError if the library does not export it
            fn.restype = res
            fn.argtypes = args
        _LIB = lib
    return _LIB


def exported_symbols():
    return sorted(SYMBOLS)


class DG:
    """One mesh + one state vector on the GPU.  Arrays are float64, shape (nz,ny,nx,N,N,N,5)."""

    def __init__(self, nx, ny, nz, p, gamma=1.4, extent=(1.0, 1.0, 1.0), device="cuda:0", brick=None, bind=True,
                 variant=None, poison=False, spacing=None, viscosity=None):
        self.lib = load_library()
        self.nx, self.ny, self.nz, self.p, self.N = nx, ny, nz, p, p + 1
        self.gamma, self.extent = float(gamma), tuple(float(e) for e in extent)
        self.shape = (nz, ny, nx, self.N, self.N, self.N, 5)
        self._h = ctypes.c_void_p()
        ext = (ctypes.c_double * 3)(*self.extent)
        rc = self.lib.dg_create(ctypes.byref(self._h), nx, ny, nz, p, self.gamma, ext)
        if rc != 0:
            self._h = None
            raise DGError(rc, f"dg_create({nx},{ny},{nz},p={p},gamma={gamma},extent={extent})")
        if brick is not None:
            self._check(self.lib.dg_set_brick(self._h, *brick))
        if variant is not None:
            self._check(self.lib.dg_set_variant(self._h, int(variant)))
        if spacing is not None:
            self._check(self.lib.dg_set_spacing(self._h, (ctypes.c_double * 3)(*[float(v) for v in spacing])))
        if viscosity is not None:     # (mu, Prandtl number): Navier-Stokes terms, dg_split_viscous / dg_rk_step_ns
            self._check(self.lib.dg_set_viscosity(self._h, float(viscosity[0]), float(viscosity[1])))
        self.workspace = None
        self.device = None
        self._torch = None
        if bind:
            self.bind(device, poison=poison)

    # -- plumbing -------------------------------------------------------------------------------
    def _check(self, rc):
        if rc != 0:
            raise DGError(rc, self.lib.dg_last_error(self._h).decode())

    def bind(self, device="cuda:0", stream=None, poison=False):
        """Allocate the workspace and hand it to the library.  poison=True fills it with 0xFF bytes (NaN as doubles)
        first: a test aid that makes any read of memory the library has not written show up in the results."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2006_15698_b200 needs a CUDA device; there is no CPU fallback")
        self.device = torch.device(device)
        self._torch = torch
        nbytes = self.lib.dg_workspace_bytes(self._h)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            if poison:
                self.workspace.fill_(255)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self._check(self.lib.dg_bind(self._h, self.workspace.data_ptr(), nbytes, self.stream.cuda_stream))

    def set_boundary(self, bc, q_inf=None):
        """bc = (x-, x+, y-, y+, z-, z+): 0 periodic, 1 slip wall, 2 far field with exterior state q_inf (5 doubles)."""
        b = (ctypes.c_int * 6)(*[int(v) for v in bc])
        qi = None if q_inf is None else (ctypes.c_double * 5)(*[float(v) for v in q_inf])
        self._check(self.lib.dg_set_boundary(self._h, b, qi))
        return self

    @property
    def state_len(self):
        return self.lib.dg_state_len(self._h)

    @property
    def workspace_bytes(self):
        return self.lib.dg_workspace_bytes(self._h)

    @property
    def launch_count(self):
        return self.lib.dg_launch_count(self._h)

    def kernel_info(self):
        out = (ctypes.c_longlong * 8)()
        self._check(self.lib.dg_kernel_info(self._h, out))
        keys = ("bx", "by", "lz", "threads", "smem_bytes", "grid", "internal_mdoubles", "variant")
        return dict(zip(keys, [int(v) for v in out]))

    def nodes(self):
        xi = np.empty(self.N)
        w = np.empty(self.N)
        self._check(self.lib.dg_nodes(self._h, xi.ctypes.data_as(_DP), w.ctypes.data_as(_DP)))
        return xi, w

    def _ptr(self, a, writable):
        """(pointer, on_device, keepalive) for a numpy array or a torch tensor of the state's size."""
        torch = self._torch
        if isinstance(a, torch.Tensor):
            if a.dtype != torch.float64 or not a.is_contiguous() or a.numel() != self.state_len:
                raise ValueError("state tensors must be contiguous float64 with dg_state_len elements")
            if a.is_cuda and a.device != self.device:
                raise ValueError("tensor is on another device")
            return ctypes.c_void_p(a.data_ptr()), int(a.is_cuda), a
        a = np.asarray(a)
        if a.dtype != np.float64 or not a.flags.c_contiguous or a.size != self.state_len:
            raise ValueError("state arrays must be C-contiguous float64 with dg_state_len elements")
        if writable and not a.flags.writeable:
            raise ValueError("output array is read-only")
        return ctypes.c_void_p(a.ctypes.data), 0, a

    def _order_before(self, dev):
        """Device tensors may have been produced on torch's current stream: make the bound stream wait for it
        (include/dg_b200.h: the library orders its work on the stream given to dg_bind only)."""
        if dev:
            cur = self._torch.cuda.current_stream(self.device)
            if cur != self.stream:
                self.stream.wait_stream(cur)

    def _order_after(self, dev):
        if dev:
            cur = self._torch.cuda.current_stream(self.device)
            if cur != self.stream:
                cur.wait_stream(self.stream)

    # -- the six calls of north_star (+ max wavespeed) ---------------------------------------------
    def set_state(self, q):
        ptr, dev, keep = self._ptr(q, False)
        self._order_before(dev)
        with self._torch.cuda.device(self.device):
            self._check(self.lib.dg_set_state(self._h, ptr, dev))
        if dev == 0 and isinstance(keep, self._torch.Tensor) and keep.is_pinned():
            self.stream.synchronize()     # the async copy reads the caller's pinned buffer
        return self

    def residual(self, out=None):
        """dQ/dt of the current state; `out` may be a numpy array, a host or a cuda tensor."""
        if out is None:
            out = np.empty(self.shape)
        ptr, dev, _ = self._ptr(out, True)
        self._order_before(dev)
        with self._torch.cuda.device(self.device):
            self._check(self.lib.dg_residual(self._h, ptr, dev))
        self._order_after(dev)
        return out

    def rk_step(self, dt, nsteps=1):
        with self._torch.cuda.device(self.device):
            self._check(self.lib.dg_rk_step(self._h, float(dt), int(nsteps)))
        return self

    def rk_step_cfl(self, cfl, nsteps=1):
        """nsteps LSERK45 steps, each with dt = cfl * min(h) / ((2p+1) * max wavespeed) of its own initial state.
        Returns (time advanced, last dt)."""
        t, dt = ctypes.c_double(0.0), ctypes.c_double(0.0)
        with self._torch.cuda.device(self.device):
            self._check(self.lib.dg_rk_step_cfl(self._h, float(cfl), int(nsteps), ctypes.byref(t), ctypes.byref(dt)))
        return t.value, dt.value

    def cfl_dt(self, cfl, lam_max):
        """dg_cfl_dt: cfl * min(h) / ((2p+1) * lam_max), formed by the library (host arithmetic, no GPU work)."""
        dt = ctypes.c_double(0.0)
        rc = self.lib.dg_cfl_dt(self._h, float(cfl), float(lam_max), ctypes.byref(dt))
        if rc != 0:
            raise DGError(rc, f"dg_cfl_dt(cfl={cfl}, lam_max={lam_max}): both must be positive and finite")
        return dt.value

    # -- block decomposition over several contexts / GPUs: face export / import, stage by stage ----------
    def rk_stage(self, dt, stage):
        with self._torch.cuda.device(self.device):
            self._check(self.lib.dg_rk_stage(self._h, float(dt), int(stage)))
        return self

    def halo_len(self, face):
        return self.lib.dg_halo_len(self._h, int(face))

    def halo_export(self, face, out=None):
        """Face traces of the current state on domain face `face` into a float64 cuda tensor (what the neighbour needs)."""
        torch = self._torch
        if out is None:
            out = torch.empty(self.halo_len(face), dtype=torch.float64, device=self.device)
        assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == self.halo_len(face)
        self._order_before(1)
        with torch.cuda.device(self.device):
            self._check(self.lib.dg_halo_export(self._h, int(face), out.data_ptr()))
        self._order_after(1)
        return out

    def set_halo(self, face, buf):
        """`buf`: float64 cuda tensor of halo_len(face) doubles the caller keeps alive and fills before every stage."""
        assert buf.is_cuda and buf.dtype == self._torch.float64 and buf.is_contiguous() and buf.numel() == self.halo_len(face)
        self._halo_keep = getattr(self, "_halo_keep", {})
        self._halo_keep[int(face)] = buf
        self._check(self.lib.dg_set_halo(self._h, int(face), buf.data_ptr()))
        return self

    def set_halo_pair(self, face, buf0, buf1):
        """Push mode: the two float64 cuda tensors the kernels read alternately for the traces beyond `face`."""
        for b in (buf0, buf1):
            assert b.is_cuda and b.dtype == self._torch.float64 and b.is_contiguous() and b.numel() == self.halo_len(face)
        self._halo_keep = getattr(self, "_halo_keep", {})
        self._halo_keep[("pair", int(face))] = (buf0, buf1)
        self._check(self.lib.dg_set_halo_pair(self._h, int(face), buf0.data_ptr(), buf1.data_ptr()))
        return self

    def set_halo_push(self, face, peer0, peer1):
        """Push mode: the neighbour's pair for its opposite face (tensors, or raw device addresses of peer-mapped memory)."""
        ptr = lambda b: int(b) if isinstance(b, int) else b.data_ptr()
        self._halo_keep = getattr(self, "_halo_keep", {})
        self._halo_keep[("push", int(face))] = (peer0, peer1)
        self._check(self.lib.dg_set_halo_push(self._h, int(face), ptr(peer0), ptr(peer1)))
        return self

    # -- paper-shaped per-kernel mode (Table II breakdown) ------------------------------------------
    def split_volume(self):
        with self._torch.cuda.device(self.device):
            self._check(self.lib.dg_split_volume(self._h))
        return self

    def split_surface(self):
        with self._torch.cuda.device(self.device):
            self._check(self.lib.dg_split_surface(self._h))
        return self

    def split_update(self, dt, stage):
        with self._torch.cuda.device(self.device):
            self._check(self.lib.dg_split_update(self._h, float(dt), int(stage)))
        return self

    def split_r(self, out=None):
        if out is None:
            out = np.empty(self.shape)
        ptr, dev, _ = self._ptr(out, True)
        with self._torch.cuda.device(self.device):
            self._check(self.lib.dg_split_get_r(self._h, ptr, dev))
        return out

    # -- viscous (Navier-Stokes) terms, SURVEY.md 8(f)-4 ---------------------------------------------
    def split_viscous(self):
        """R += div Fv(Q, grad Q) (after split_volume + split_surface: R = L(Q) + div Fv)."""
        with self._torch.cuda.device(self.device):
            self._check(self.lib.dg_split_viscous(self._h))
        return self

    def residual_ns(self, out=None):
        """dQ/dt = L(Q) + div Fv of the current state (volume, surface and viscous kernels, then the copy out)."""
        return self.split_volume().split_surface().split_viscous().split_r(out)

    def rk_step_ns(self, dt, nsteps=1):
        with self._torch.cuda.device(self.device):
            self._check(self.lib.dg_rk_step_ns(self._h, float(dt), int(nsteps)))
        return self

    def rk_step_split(self, dt, nsteps=1):
        """nsteps LSERK45 steps as 5 x (volume, surface, update-project) launches."""
        for _ in range(int(nsteps)):
            for stage in range(5):
                self.split_volume().split_surface().split_update(dt, stage)
        return self

    def get_state(self, out=None):
        if out is None:
            out = np.empty(self.shape)
        ptr, dev, _ = self._ptr(out, True)
        self._order_before(dev)
        with self._torch.cuda.device(self.device):
            self._check(self.lib.dg_get_state(self._h, ptr, dev))
        self._order_after(dev)
        return out

    def max_wavespeed(self):
        lam = ctypes.c_double(0.0)
        with self._torch.cuda.device(self.device):
            self._check(self.lib.dg_max_wavespeed(self._h, ctypes.byref(lam)))
        return lam.value

    def close(self):
        if getattr(self, "_h", None):
            if self.workspace is not None:
                self._torch.cuda.synchronize(self.device)
            self.lib.dg_destroy(self._h)
            self._h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

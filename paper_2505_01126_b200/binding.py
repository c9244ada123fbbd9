"""Thin ctypes binding of ``libacclb.so`` (include/acclb.h): argument marshalling only.

Every step of the path runs in the hand-written sm_100a kernels of ``csrc/``; PyTorch provides device memory
(the workspace block and the field tensors) and the stream.  There is no CPU fallback: ``load()`` raises when
the library is missing and every call needs a CUDA device.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libacclb.so"
HEADER = _PKG.parent / "include" / "acclb.h"

NDIAG = 9
NKERNELS = 12
KERNEL_NAMES = ("unused0", "k_lb", "unused2", "k_init", "k_moments", "k_diagnostics", "k_lb_tp", "k_seam",
                "k_advect", "k_geom_r", "k_mr_step", "k_lb_tp_stage")
DIAG_NAMES = ("ke", "dissipation", "sum_phi", "sum_pstar", "sum_mx", "sum_my", "sum_mz", "umax", "step")
ERRORS = {0: "ACCLB_OK", -1: "ACCLB_EINVAL", -2: "ACCLB_EWORKSPACE", -3: "ACCLB_ECUDA", -4: "ACCLB_ENUMERIC"}

SYMBOLS = ("accLB_workspace_bytes", "accLB_create", "accLB_init", "accLB_step", "accLB_moments",
           "accLB_diagnostics", "accLB_run_host", "accLB_launch_count", "accLB_profile",
           "accLB_profile_read", "accLB_set_variant", "accLB_halo_chunks", "accLB_destroy",
           "accLB_last_error", "accLB_stats_increments", "accLB_stats_pdf", "accLB_stats_spectrum",
           "accLB_stats_increments_static")


class Params(C.Structure):
    """Mirror of ``accLB_params``."""
    _fields_ = [
        ("tau", C.c_double),
        ("two_phase", C.c_int),
        ("rho_l", C.c_double), ("rho_g", C.c_double),
        ("sigma", C.c_double), ("mobility", C.c_double), ("width", C.c_double),
        ("force_type", C.c_int), ("force_amp", C.c_double), ("force_k", C.c_int),
        ("store_fp32", C.c_int), ("host_staging", C.c_int),
        ("device", C.c_int), ("stream", C.c_void_p),
        ("gravity", C.c_double * 3), ("rho_ref", C.c_double), ("phi_integrator", C.c_int),
        ("moment_storage", C.c_int),
        ("halo_z", C.c_int), ("z_origin", C.c_int), ("nz_global", C.c_int),
    ]


class HaloChunk(C.Structure):
    """Mirror of ``accLB_halo_chunk``."""
    _fields_ = [("ptr", C.c_void_p), ("bytes", C.c_size_t), ("side", C.c_int), ("dir", C.c_int)]


MAX_HALO_CHUNKS = 16


class AccLBError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"{ERRORS.get(code, code)}: {text}")
        self.code = code


_lib = None
_dp = C.c_void_p  # raw device / host addresses


def load():
    """dlopen libacclb.so; raise (never fall back) when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2505_01126_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(str(LIB_PATH))
    L.accLB_workspace_bytes.restype = C.c_size_t
    L.accLB_workspace_bytes.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(Params)]
    L.accLB_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.POINTER(Params), C.c_void_p, C.c_size_t]
    L.accLB_init.argtypes = [C.c_void_p, _dp, _dp, _dp]
    L.accLB_step.argtypes = [C.c_void_p, C.c_int]
    L.accLB_moments.argtypes = [C.c_void_p, _dp, _dp, _dp]
    L.accLB_diagnostics.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.c_int]
    L.accLB_run_host.argtypes = [C.c_void_p, _dp, _dp, _dp, C.c_int, _dp, _dp, _dp, C.POINTER(C.c_double)]
    L.accLB_launch_count.restype = C.c_longlong
    L.accLB_launch_count.argtypes = [C.c_void_p]
    L.accLB_profile.argtypes = [C.c_void_p, C.c_int]
    L.accLB_profile_read.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_longlong), C.c_int]
    L.accLB_set_variant.argtypes = [C.c_void_p, C.c_int]
    L.accLB_halo_chunks.argtypes = [C.c_void_p, C.c_int, C.POINTER(HaloChunk), C.c_int]
    L.accLB_destroy.argtypes = [C.c_void_p]
    L.accLB_last_error.restype = C.c_char_p
    L.accLB_stats_increments.argtypes = [_dp, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int), C.c_int, C.POINTER(C.c_double), _dp,
                                         C.c_size_t, C.c_int, C.c_void_p]
    L.accLB_stats_pdf.argtypes = [_dp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int,
                                  C.POINTER(C.c_ulonglong), _dp, C.c_size_t, C.c_int, C.c_void_p]
    L.accLB_stats_spectrum.argtypes = [_dp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_double), _dp, C.c_size_t,
                                       C.c_int, C.c_void_p]
    L.accLB_stats_increments_static.argtypes = [_dp, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int), C.c_int, C.POINTER(C.c_double),
                                                C.c_int, C.c_void_p]
    _lib = L
    return L


def _check(code):
    if code != 0:
        raise AccLBError(code, load().accLB_last_error().decode())


def make_params(*, tau, two_phase=0, rho_l=1.0, rho_g=1.0, sigma=0.0, mobility=0.0, width=4.0, force_type=0,
                force_amp=0.0, force_k=1, store_fp32=0, host_staging=0, device=0, stream=None,
                gravity=(0.0, 0.0, 0.0), rho_ref=0.0, phi_rk3=0, moment_storage=0, halo_z=0, z_origin=0, nz_global=0):
    return Params(tau, int(two_phase), rho_l, rho_g, sigma, mobility, width, int(force_type), force_amp, int(force_k),
                  int(store_fp32), int(host_staging), int(device), stream, (C.c_double * 3)(*gravity), rho_ref,
                  int(phi_rk3), int(moment_storage), int(halo_z), int(z_origin), int(nz_global))


def workspace_bytes(nx, ny, nz, params):
    return load().accLB_workspace_bytes(nx, ny, nz, C.byref(params))


class AccLB:
    """One periodic box on one GPU.  Fields are fp64 CUDA tensors: scalars [nz][ny][nx], vectors [3][nz][ny][nx]."""

    def __init__(self, nx, ny, nz, *, device=0, stream=None, workspace=None, **params):
        import torch

        L = load()
        self._torch = torch
        self.device = torch.device("cuda", device)
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        self.stream = stream
        self.params = make_params(device=device, stream=stream.cuda_stream, **params)
        self.shape = (nz, ny, nx)
        self.nx, self.ny, self.nz = nx, ny, nz
        self.n = nx * ny * nz
        self.two_phase = bool(self.params.two_phase)
        nbytes = L.accLB_workspace_bytes(nx, ny, nz, C.byref(self.params))
        if nbytes == 0:
            raise AccLBError(-1, f"invalid grid {nx}x{ny}x{nz} or parameters")
        if workspace is None:
            workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)  # torch owns device memory
        assert workspace.is_cuda and workspace.dtype == torch.uint8 and workspace.is_contiguous() and workspace.numel() >= nbytes
        self.workspace = workspace  # (a caller-provided block, e.g. a view into a larger tensor, is used as it is)
        self.workspace_bytes = nbytes
        h = C.c_void_p()
        _check(L.accLB_create(C.byref(h), nx, ny, nz, C.byref(self.params), self.workspace.data_ptr(), nbytes))
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            load().accLB_destroy(self._h)
            self._h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _dev(self, t, shape):
        torch = self._torch
        assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == tuple(shape), \
            (t.device, t.dtype, tuple(t.shape), shape)
        return t.data_ptr()

    def _on_stream(self):
        """The context enqueues on the stream it was created with; the caller's tensors must be ordered on the same one."""
        cur = self._torch.cuda.current_stream(self.device)
        assert cur.cuda_stream == self.stream.cuda_stream, \
            "AccLB was created on another stream: call it under `with torch.cuda.stream(sim.stream)` (or synchronise)"

    def init(self, rho, u, phi=None):
        self._on_stream()
        _check(load().accLB_init(self._h, self._dev(rho, self.shape), self._dev(u, (3,) + self.shape),
                                 self._dev(phi, self.shape) if phi is not None else None))

    def step(self, nsteps=1):
        _check(load().accLB_step(self._h, int(nsteps)))

    def moments(self, rho=None, u=None, phi=None):
        self._on_stream()
        torch = self._torch
        kw = dict(dtype=torch.float64, device=self.device)
        rho = torch.empty(self.shape, **kw) if rho is None else rho
        u = torch.empty((3,) + self.shape, **kw) if u is None else u
        if self.two_phase and phi is None:
            phi = torch.empty(self.shape, **kw)
        _check(load().accLB_moments(self._h, self._dev(rho, self.shape), self._dev(u, (3,) + self.shape),
                                    self._dev(phi, self.shape) if self.two_phase else None))
        return rho, u, (phi if self.two_phase else None)

    def diagnostics(self):
        out = (C.c_double * NDIAG)()
        _check(load().accLB_diagnostics(self._h, out, NDIAG))
        return dict(zip(DIAG_NAMES, list(out)))

    def run_host(self, rho, u, phi, nsteps, rho_out=None, u_out=None, phi_out=None, diag=True):
        """Host-buffer path: CPU tensors (pinned for asynchronous copies) in and out."""
        self._on_stream()
        def hp(t, shape):
            if t is None:
                return None
            assert (not t.is_cuda) and t.dtype == self._torch.float64 and t.is_contiguous() and tuple(t.shape) == tuple(shape)
            return t.data_ptr()
        d = (C.c_double * NDIAG)() if diag else None
        _check(load().accLB_run_host(self._h, hp(rho, self.shape), hp(u, (3,) + self.shape), hp(phi, self.shape),
                                     int(nsteps), hp(rho_out, self.shape), hp(u_out, (3,) + self.shape),
                                     hp(phi_out, self.shape), d))
        return dict(zip(DIAG_NAMES, list(d))) if diag else None

    def profile(self, enable=True):
        _check(load().accLB_profile(self._h, int(bool(enable))))

    def profile_read(self):
        """{kernel: (total ms, launches)} since the last read; synchronises."""
        ms = (C.c_double * NKERNELS)()
        cnt = (C.c_longlong * NKERNELS)()
        _check(load().accLB_profile_read(self._h, ms, cnt, NKERNELS))
        return {k: (ms[i], cnt[i]) for i, k in enumerate(KERNEL_NAMES)}

    def set_variant(self, v):
        _check(load().accLB_set_variant(self._h, int(v)))

    def halo_chunks(self, full=False):
        """The halo exchange of a z-slab context for its CURRENT buffers: a list of (view, side, dir), `view` a uint8 view
        into the workspace (no copy), side -1 / +1 the z-neighbour, dir 0 = send, 1 = receive (include/acclb.h)."""
        arr = (HaloChunk * MAX_HALO_CHUNKS)()
        n = load().accLB_halo_chunks(self._h, int(bool(full)), arr, MAX_HALO_CHUNKS)
        if n < 0:
            _check(n)
        base = self.workspace.data_ptr()
        out = []
        for c in arr[:n]:
            off = c.ptr - base
            assert 0 <= off and off + c.bytes <= self.workspace.numel()
            out.append((self.workspace[off:off + c.bytes], c.side, c.dir))
        return out

    @property
    def launch_count(self):
        return int(load().accLB_launch_count(self._h))


# ---------------------------------------------------------------------------------------- turbulence statistics (8(f) #4)
def _stats_common(t, ndim):
    import torch
    assert t.is_cuda and t.is_contiguous() and t.dim() == ndim, (t.device, tuple(t.shape))
    dev = t.device
    return torch, dev, torch.cuda.current_stream(dev).cuda_stream


def stats_increments(u, separations):
    """S_p(r), p = 2, 3, 4, of the longitudinal velocity increments of u [3][nz][ny][nx] (CUDA fp64): array [nr][3]."""
    torch, dev, stream = _stats_common(u, 4)
    assert u.dtype == torch.float64 and u.shape[0] == 3
    _, nz, ny, nx = u.shape
    nr = len(separations)
    r = (C.c_int * nr)(*[int(v) for v in separations])
    out = (C.c_double * (3 * nr))()
    scratch = torch.empty(3 * nr, dtype=torch.float64, device=dev)
    _check(load().accLB_stats_increments(u.data_ptr(), nx, ny, nz, r, nr, out, scratch.data_ptr(), scratch.numel() * 8,
                                         dev.index or 0, stream))
    return [[out[3 * j + p] for p in range(3)] for j in range(nr)]


STATS_STATIC_MAX_NR = 64


def stats_increments_static(u, separations):
    """stats_increments through the entry point that allocates nothing: the accumulators are a fixed array inside the library
    (at most STATS_STATIC_MAX_NR separations; calls on one device share it and must not overlap).  Array [nr][3]."""
    torch, dev, stream = _stats_common(u, 4)
    assert u.dtype == torch.float64 and u.shape[0] == 3
    _, nz, ny, nx = u.shape
    nr = len(separations)
    r = (C.c_int * nr)(*[int(v) for v in separations])
    out = (C.c_double * (3 * nr))()
    _check(load().accLB_stats_increments_static(u.data_ptr(), nx, ny, nz, r, nr, out, dev.index or 0, stream))
    return [[out[3 * j + p] for p in range(3)] for j in range(nr)]


def stats_pdf(u, r, scale, lo, hi, nbins):
    """Histogram (nbins counts) of the longitudinal increments at separation r, divided by scale, on [lo, hi)."""
    torch, dev, stream = _stats_common(u, 4)
    assert u.dtype == torch.float64 and u.shape[0] == 3
    _, nz, ny, nx = u.shape
    counts = (C.c_ulonglong * nbins)()
    scratch = torch.empty(nbins, dtype=torch.int64, device=dev)
    _check(load().accLB_stats_pdf(u.data_ptr(), nx, ny, nz, int(r), float(scale), float(lo), float(hi), int(nbins), counts,
                                  scratch.data_ptr(), scratch.numel() * 8, dev.index or 0, stream))
    return list(counts)


def stats_spectrum(uhat, nx, nshell):
    """Shell sums E[k] of uhat = rfftn of ncomp real fields, [ncomp][nz][ny][nx/2+1] complex128 (the caller's FFT)."""
    torch, dev, stream = _stats_common(uhat, 4)
    assert uhat.dtype == torch.complex128 and uhat.shape[3] == nx // 2 + 1
    ncomp, nz, ny, _ = uhat.shape
    E = (C.c_double * nshell)()
    scratch = torch.empty(nshell, dtype=torch.float64, device=dev)
    _check(load().accLB_stats_spectrum(uhat.data_ptr(), nx, ny, nz, ncomp, int(nshell), E, scratch.data_ptr(),
                                       scratch.numel() * 8, dev.index or 0, stream))
    return list(E)

"""Thin ctypes binding of include/flatspin.h -- argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/flatspin.cu.  torch is used for device
memory (tensors own the buffers whose pointers cross the C ABI) and for the stream.  There is no CPU
fallback: if the shared library is missing or no CUDA device is present, construction raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

from . import build as _build

FS_OK, FS_ERR_ARG, FS_ERR_COINCIDENT, FS_ERR_WORKSPACE, FS_ERR_CUDA, FS_ERR_MAXFLIPS = 0, -1, -2, -3, -4, -5
FIELD_TOTAL, FIELD_DIP, FIELD_EXT, FIELD_THERMAL = 0, 1, 2, 3
GATHER_AUTO, GATHER_ELL_F64, GATHER_STENCIL, GATHER_STENCIL_PLAIN, GATHER_STENCIL_F32 = 0, 1, 2, 3, 4

EXPORTS = [
    "fs_workspace_bytes", "fs_create", "fs_create_ensemble", "fs_destroy", "fs_get_info", "fs_set_spins",
    "fs_get_spins", "fs_set_thermal", "fs_set_field", "fs_set_field_ensemble", "fs_set_gather_variant",
    "fs_update_fields", "fs_scan", "fs_scan_ensemble", "fs_relax", "fs_relax_ensemble", "fs_get_counters",
    "fs_get_fields", "fs_get_flip_log", "fs_get_neighbors", "fs_step_host", "fs_relax_host",
    "fs_kernel_launches", "fs_last_error", "fs_get_lattice", "fs_measure_fp64_peak", "fs_sweep", "fs_sweep_anneal", "fs_set_local_field",
    "fs_set_batch", "fs_get_batch_stats", "fs_sweep_ex", "fs_correlation", "fs_vertex_populations", "fs_get_flip_log_window",
    "fs_measure_fp32_peak", "fs_scan_static",
]
SCAN_STATIC_MAX_N = 4194304          # FS_SCAN_STATIC_MAX_N of include/flatspin.h


class FsParams(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("alpha", "b", "c", "beta", "gamma", "neighbor_distance")]


class FlatspinError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"flatspin error {code}: {msg}")
        self.code = code


_lib = None


def load_library(path: str | None = None):
    """dlopen libflatspin_b200.so and declare the prototypes.  Fails loudly if it is missing."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or _build.LIB
    if not os.path.exists(path):
        raise FileNotFoundError(f"{path} not built: run `python -c 'import __graft_entry__ as g; g.build()'`")
    L = C.CDLL(path)
    vp, i64, i32, dbl, P = C.c_void_p, C.c_int64, C.c_int32, C.c_double, C.POINTER
    sig = {
        "fs_workspace_bytes": [i64, i32, vp, P(FsParams), P(C.c_size_t), vp],
        "fs_create": [P(vp), i64, vp, vp, vp, P(FsParams), vp, C.c_size_t, vp],
        "fs_create_ensemble": [P(vp), i64, i32, vp, vp, vp, P(FsParams), vp, C.c_size_t, vp],
        "fs_destroy": [vp],
        "fs_get_info": [vp, P(i64), P(i32), P(i32), P(i64)],
        "fs_set_spins": [vp, vp], "fs_get_spins": [vp, vp],
        "fs_set_thermal": [vp, dbl, C.c_uint64],
        "fs_set_field": [vp, dbl, dbl, C.c_uint32],
        "fs_set_field_ensemble": [vp, vp, C.c_uint32],
        "fs_set_gather_variant": [vp, i32],
        "fs_update_fields": [vp],
        "fs_scan": [vp, P(i64), P(i64), P(dbl)],
        "fs_scan_ensemble": [vp, vp, vp, vp],
        "fs_relax": [vp, i64, P(i64)],
        "fs_relax_ensemble": [vp, i64, vp],
        "fs_get_counters": [vp, vp, vp, i32],
        "fs_get_fields": [vp, i32, vp],
        "fs_get_flip_log": [vp, i32, vp, i64, P(i64)],
        "fs_get_neighbors": [vp, vp, P(i32)],
        "fs_step_host": [vp, vp, vp, P(i64), P(i64), P(dbl)],
        "fs_relax_host": [vp, dbl, dbl, C.c_uint32, vp, P(i64)],
        "fs_kernel_launches": [],
        "fs_last_error": [],
        "fs_get_lattice": [vp, vp, vp],
        "fs_sweep": [vp, vp, i32, C.c_uint32, vp, i64, vp],
        "fs_set_local_field": [vp, vp],
        "fs_sweep_anneal": [vp, vp, vp, i32, C.c_uint32, vp, i64, vp],
        "fs_measure_fp64_peak": [P(dbl), vp],
        "fs_measure_fp32_peak": [P(dbl), vp],
        "fs_set_batch": [vp, i32, i32],
        "fs_sweep_ex": [vp, vp, vp, vp, vp, i32, C.c_uint32, vp, i64, vp],
        "fs_correlation": [vp, dbl, i32, vp, vp],
        "fs_vertex_populations": [vp, vp, i64, vp],
        "fs_get_flip_log_window": [vp, i32, vp, i64, P(i64), P(i64)],
        "fs_get_batch_stats": [vp, vp],
        "fs_scan_static": [i64, vp, vp, vp, vp, P(FsParams), dbl, dbl, dbl, C.c_uint64, C.c_uint32, vp, vp],
    }
    for name, args in sig.items():
        fn = getattr(L, name)
        fn.argtypes = args
        fn.restype = C.c_int
    L.fs_kernel_launches.restype = C.c_int64
    L.fs_last_error.restype = C.c_char_p
    if path == _build.LIB:
        _lib = L
    return L


def _check(L, rc, allow=()):
    if rc != FS_OK and rc not in allow:
        raise FlatspinError(rc, L.fs_last_error().decode())
    return rc


def kernel_launches() -> int:
    return int(load_library().fs_kernel_launches())


def measure_fp64_peak(stream=None) -> float:
    """DFMA/s of the DFMA-chain calibration kernel (the FP64 roofline denominator)."""
    L = load_library()
    v = C.c_double()
    sp = C.c_void_p(stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream)
    _check(L, L.fs_measure_fp64_peak(C.byref(v), sp))
    return float(v.value)


def measure_fp32_peak(stream=None) -> float:
    """FFMA/s of the FFMA-chain calibration kernel (denominator of the optional fp32 field path)."""
    L = load_library()
    v = C.c_double()
    sp = C.c_void_p(stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream)
    _check(L, L.fs_measure_fp32_peak(C.byref(v), sp))
    return float(v.value)


def scan_static(angle, hc, s, hdip, params: dict, hx, hy, sigma_th=0.0, seed=0, step=0, result=None, stream=None):
    """fs_scan_static: the switching scan without a handle, a workspace or any device allocation inside the library
    (for programs whose own pool holds the card's memory, or that cannot take cudaMalloc's device-wide stall).  All
    arguments are CUDA tensors the caller owns: angle [N] f64, hc [N] f64, s [N] int8, hdip [N,2] f64; `result` is
    a 3-element int64 tensor (allocated here with torch if None; pass your own to keep this call allocation-free
    on the Python side too).  Asynchronous; returns `result`: [n_switchable, best_index, bits of best_L] -- read the
    last one with result[2:3].view(torch.float64).  N <= SCAN_STATIC_MAX_N, else FlatspinError(FS_ERR_ARG)."""
    L = load_library()
    for t, dt in ((angle, torch.float64), (hc, torch.float64), (s, torch.int8), (hdip, torch.float64)):
        assert t.is_cuda and t.is_contiguous() and t.dtype == dt
    N = int(angle.shape[0])
    assert hc.numel() == N and s.numel() == N and hdip.numel() == 2 * N
    if result is None:
        result = torch.empty(3, dtype=torch.int64, device=angle.device)
    assert result.is_cuda and result.dtype == torch.int64 and result.numel() >= 3
    p = FsParams(*[float(params.get(k, 1.0)) for k in ("alpha", "b", "c", "beta", "gamma", "neighbor_distance")])
    with torch.cuda.device(angle.device):
        sp = C.c_void_p(stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream)
        _check(L, L.fs_scan_static(N, angle.data_ptr(), hc.data_ptr(), s.data_ptr(), hdip.data_ptr(), C.byref(p),
                                   float(hx), float(hy), float(sigma_th), int(seed), int(step), result.data_ptr(), sp))
    return result


class Sim:
    """One simulation handle (R >= 1 replicas).  Mirrors the fs_* entry points one to one."""

    def __init__(self, pos, angle, hc, params: dict, device="cuda:0", stream: torch.cuda.Stream | None = None):
        if not torch.cuda.is_available():
            raise RuntimeError("flatspin_b200 needs a CUDA device; there is no CPU fallback")
        self.L = load_library()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._sp = C.c_void_p(self.stream.cuda_stream)
        f64 = dict(dtype=torch.float64, device=self.device)
        with torch.cuda.stream(self.stream):
            pos_d = torch.as_tensor(np.ascontiguousarray(pos, np.float64)).to(**f64).contiguous()
            ang_d = torch.as_tensor(np.ascontiguousarray(angle, np.float64)).to(**f64).contiguous()
            hc_np = np.ascontiguousarray(hc, np.float64)
            hc_d = torch.as_tensor(hc_np).to(**f64).contiguous()
        self.N = int(ang_d.shape[0])
        self.R = 1 if hc_np.ndim == 1 else int(hc_np.shape[0])
        assert pos_d.shape == (self.N, 2) and hc_d.numel() == self.R * self.N
        self.params = FsParams(*[float(params[k]) for k in ("alpha", "b", "c", "beta", "gamma", "neighbor_distance")])
        nbytes = C.c_size_t(0)
        _check(self.L, self.L.fs_workspace_bytes(self.N, self.R, pos_d.data_ptr(), C.byref(self.params),
                                                 C.byref(nbytes), self._sp))
        self.workspace_bytes = int(nbytes.value)
        self.workspace = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        self._ws_ptr = (base + 255) // 256 * 256
        h = C.c_void_p()
        _check(self.L, self.L.fs_create_ensemble(C.byref(h), self.N, self.R, pos_d.data_ptr(), ang_d.data_ptr(),
                                                 hc_d.data_ptr(), C.byref(self.params), self._ws_ptr,
                                                 self.workspace_bytes, self._sp))
        self.h = h
        n, r, k, i = C.c_int64(), C.c_int32(), C.c_int32(), C.c_int64()
        _check(self.L, self.L.fs_get_info(self.h, C.byref(n), C.byref(r), C.byref(k), C.byref(i)))
        self.K, self.n_interactions = int(k.value), int(i.value)

    def close(self):
        if getattr(self, "h", None):
            self.L.fs_destroy(self.h)
            self.h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- state
    def set_spins(self, s):
        t = s if isinstance(s, torch.Tensor) else torch.as_tensor(np.ascontiguousarray(s, np.int8))
        t = t.to(device=self.device, dtype=torch.int8).contiguous()
        assert t.numel() == self.R * self.N
        _check(self.L, self.L.fs_set_spins(self.h, t.data_ptr()))
        self.stream.synchronize()   # `t` may be a temporary

    def get_spins(self) -> torch.Tensor:
        out = torch.empty((self.R, self.N) if self.R > 1 else (self.N,), dtype=torch.int8, device=self.device)
        _check(self.L, self.L.fs_get_spins(self.h, out.data_ptr()))
        return out

    def set_thermal(self, sigma_th, seed):
        _check(self.L, self.L.fs_set_thermal(self.h, float(sigma_th), int(seed)))

    def set_field(self, hx, hy, step=0):
        _check(self.L, self.L.fs_set_field(self.h, float(hx), float(hy), int(step)))

    def set_field_ensemble(self, h, step=0):
        h = np.ascontiguousarray(h, np.float64); assert h.shape == (self.R, 2)
        _check(self.L, self.L.fs_set_field_ensemble(self.h, h.ctypes.data, int(step)))

    def set_local_field(self, h):
        """Per-spin external field [N,2] added to the global one; None clears it."""
        if h is None:
            _check(self.L, self.L.fs_set_local_field(self.h, None)); return
        t = torch.as_tensor(np.ascontiguousarray(h, np.float64)).to(self.device).contiguous()
        assert tuple(t.shape) == (self.N, 2)
        _check(self.L, self.L.fs_set_local_field(self.h, t.data_ptr()))
        self.stream.synchronize()

    def set_gather_variant(self, v):
        _check(self.L, self.L.fs_set_gather_variant(self.h, int(v)))

    def set_batch(self, max_seeds, seq_threshold=64):
        """Exact batched flips: seeds per round (0 = off) and the candidate count below which k_relax takes over."""
        _check(self.L, self.L.fs_set_batch(self.h, int(max_seeds), int(seq_threshold)))

    def batch_stats(self) -> dict:
        out = np.zeros(4, np.int64)
        _check(self.L, self.L.fs_get_batch_stats(self.h, out.ctypes.data))
        return {"max_seeds": int(out[0]), "flips": int(out[1]), "rounds": int(out[2]), "seq_threshold": int(out[3])}

    def lattice(self) -> dict:
        info = np.zeros(12, np.int32); d = np.zeros(2, np.float64)
        _check(self.L, self.L.fs_get_lattice(self.h, info.ctypes.data, d.ctypes.data))
        keys = ("active", "reason", "nsub", "U", "V", "Ru", "Rv", "slots", "warps_per_cta", "smem_bytes", "inversion_pairs", "row_pairs")
        out = {k: int(v) for k, v in zip(keys, info)}
        out["active"] = bool(out["active"]); out["inversion_pairs"] = bool(out["inversion_pairs"]); out["max_dev"] = float(d[0]); out["w_max"] = float(d[1])
        return out

    # ---- compute
    def update_fields(self):
        _check(self.L, self.L.fs_update_fields(self.h))

    def scan(self):
        n, b, l = C.c_int64(), C.c_int64(), C.c_double()
        _check(self.L, self.L.fs_scan(self.h, C.byref(n), C.byref(b), C.byref(l)))
        return int(n.value), int(b.value), float(l.value)

    def scan_async(self):
        _check(self.L, self.L.fs_scan(self.h, None, None, None))

    def scan_ensemble(self):
        n = np.zeros(self.R, np.int64); b = np.zeros(self.R, np.int64); l = np.zeros(self.R, np.float64)
        _check(self.L, self.L.fs_scan_ensemble(self.h, n.ctypes.data, b.ctypes.data, l.ctypes.data))
        return n, b, l

    def relax(self, max_flips=0, sync=True):
        if not sync:
            _check(self.L, self.L.fs_relax(self.h, int(max_flips), None))
            return None
        n = C.c_int64()
        _check(self.L, self.L.fs_relax(self.h, int(max_flips), C.byref(n)), allow=(FS_ERR_MAXFLIPS,))
        return int(n.value)

    def sweep(self, fields, step0=0, per_step=True, max_flips=0, sync=True, sigma=None, local_scale=None, local_series=None):
        """Whole protocol in one launch.  fields [T,2]; sigma [T] = thermal std per step (annealing) or None;
        local_scale [T] scales the static per-spin field per step, local_series [T,N,2] adds a per-spin field per step.
        Returns (flips per replica [R] or None if not sync, flips per step tensor [R,T] on the device or None)."""
        def dev(a):
            return None if a is None else torch.as_tensor(np.ascontiguousarray(a, np.float64)).to(self.device)
        f = dev(fields)
        T = int(f.shape[0])
        sg, ls, lser = dev(sigma), dev(local_scale), dev(local_series)
        assert sg is None or sg.numel() == T
        assert ls is None or ls.numel() == T
        assert lser is None or tuple(lser.shape) == (T, self.N, 2)
        ps = torch.zeros((self.R, T), dtype=torch.int64, device=self.device) if per_step else None
        n = np.zeros(self.R, np.int64)
        ptr = lambda t: None if t is None else t.data_ptr()
        _check(self.L, self.L.fs_sweep_ex(self.h, f.data_ptr(), ptr(sg), ptr(ls), ptr(lser), T, int(step0),
                                          ps.data_ptr() if per_step else None, int(max_flips),
                                          n.ctypes.data if sync else None), allow=(FS_ERR_MAXFLIPS,))
        if not sync:
            self._keep = (f, sg, ls, lser)                 # the kernel reads them asynchronously
        return (n if sync else None), ps

    def correlation(self, bin_width, nbins):
        """Spin-spin correlation by separation: (sum of c_ij [R,nbins] or [nbins], pairs per bin [nbins])."""
        sm = torch.zeros((self.R, int(nbins)), dtype=torch.int64, device=self.device)
        cnt = torch.zeros(int(nbins), dtype=torch.int64, device=self.device)
        _check(self.L, self.L.fs_correlation(self.h, float(bin_width), int(nbins), sm.data_ptr(), cnt.data_ptr()))
        return (sm if self.R > 1 else sm[0]), cnt

    def vertex_populations(self, vertices):
        """Counts of Type I..IV vertices ([R,4] or [4]); vertices [V,4] spin indices."""
        v = torch.as_tensor(np.ascontiguousarray(vertices, np.int32)).to(self.device)
        assert v.dim() == 2 and v.shape[1] == 4
        out = torch.zeros((self.R, 4), dtype=torch.int64, device=self.device)
        _check(self.L, self.L.fs_vertex_populations(self.h, v.data_ptr(), int(v.shape[0]), out.data_ptr()))
        self.stream.synchronize()                          # `v` may be a temporary
        return out if self.R > 1 else out[0]

    def relax_ensemble(self, max_flips=0):
        n = np.zeros(self.R, np.int64)
        _check(self.L, self.L.fs_relax_ensemble(self.h, int(max_flips), n.ctypes.data), allow=(FS_ERR_MAXFLIPS,))
        return n

    def counters(self, reset=False):
        tot = np.zeros(self.R, np.int64); last = np.zeros(self.R, np.int64)
        _check(self.L, self.L.fs_get_counters(self.h, tot.ctypes.data, last.ctypes.data, int(reset)))
        return tot, last

    def get_fields(self, which=FIELD_TOTAL) -> torch.Tensor:
        shape = (self.R, self.N, 2) if self.R > 1 else (self.N, 2)
        out = torch.empty(shape, dtype=torch.float64, device=self.device)
        _check(self.L, self.L.fs_get_fields(self.h, int(which), out.data_ptr()))
        return out

    def get_flip_log(self, replica=0, cap=None) -> torch.Tensor:
        cap = int(cap if cap is not None else 4 * self.N + 1024)
        out = torch.empty(cap, dtype=torch.int32, device=self.device)
        n = C.c_int64()
        first = C.c_int64()
        _check(self.L, self.L.fs_get_flip_log_window(self.h, int(replica), out.data_ptr(), cap, C.byref(n), C.byref(first)))
        self.last_log_count = int(n.value); self.last_log_first = int(first.value)
        return out[:min(int(n.value) - int(first.value), cap)]

    def get_neighbors(self) -> torch.Tensor:
        out = torch.empty((self.N, max(self.K, 1)), dtype=torch.int32, device=self.device)
        k = C.c_int32()
        _check(self.L, self.L.fs_get_neighbors(self.h, out.data_ptr(), C.byref(k)))
        return out[:, :self.K]

    # ---- host-buffer entry points (end-to-end timing)
    def step_host(self, s_host: torch.Tensor, h_host_out: torch.Tensor | None):
        assert s_host.dtype == torch.int8 and not s_host.is_cuda and s_host.numel() == self.R * self.N
        assert h_host_out is None or (h_host_out.dtype == torch.float64 and not h_host_out.is_cuda and h_host_out.numel() == 2 * self.R * self.N)
        n, b, l = C.c_int64(), C.c_int64(), C.c_double()
        _check(self.L, self.L.fs_step_host(self.h, s_host.data_ptr(), h_host_out.data_ptr() if h_host_out is not None else None,
                                           C.byref(n), C.byref(b), C.byref(l)))
        return int(n.value), int(b.value), float(l.value)

    def relax_host(self, hx, hy, step, s_host_out: torch.Tensor):
        assert s_host_out.dtype == torch.int8 and not s_host_out.is_cuda and s_host_out.numel() == self.R * self.N
        n = C.c_int64()
        _check(self.L, self.L.fs_relax_host(self.h, float(hx), float(hy), int(step), s_host_out.data_ptr(), C.byref(n)))
        return int(n.value)

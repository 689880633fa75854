"""Thin ctypes binding of include/agnvar.h (libagnvar.so).

Argument marshalling only: every step of the path runs in the CUDA kernels behind the C ABI.
PyTorch is used for device memory (tensors own every buffer, including the workspace) and for the
current CUDA stream.  There is no CPU fallback: if the library is missing or cannot be loaded the
import of a symbol raises.
"""
import ctypes as C
import os

import torch

from . import _build

AGNVAR_F32, AGNVAR_F64 = 0, 1
AGNVAR_ERDF_BPL, AGNVAR_ERDF_LOGNORMAL = 0, 1
(OP_ERDF_SAMPLE_SORTED, OP_TK_GENERATE, OP_E13_ITERATE, OP_PERIODOGRAM, OP_STRUCTURE_FUNCTION, OP_DELTA_M_PROB,
 OP_ENSEMBLE_SF, OP_SLICE_SAMPLE_SORTED) = 1, 2, 3, 4, 5, 6, 7, 8

EXPORTS = (
    "agnvar_workspace_bytes", "agnvar_psd_bpl", "agnvar_erdf_sample_sorted", "agnvar_erdf_table", "agnvar_tk_generate",
    "agnvar_e13_iterate", "agnvar_periodogram", "agnvar_philox_u32", "agnvar_strerror", "agnvar_version",
    "agnvar_launch_count", "agnvar_trace_begin", "agnvar_trace_end", "agnvar_kernel_name",
    "agnvar_structure_function", "agnvar_delta_m_prob", "agnvar_ensemble_sf", "agnvar_moments",
    "agnvar_slice_sample_sorted",
    "agnvar_static_scratch_bytes", "agnvar_structure_function_static_bytes", "agnvar_structure_function_static",
)


class AgnvarError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        super().__init__(f"{where}: agnvar status {status} ({strerror(status)})")


class agnvar_psd(C.Structure):
    _fields_ = [("A", C.c_double), ("f_b", C.c_double), ("alpha_low", C.c_double), ("alpha_high", C.c_double)]


class agnvar_erdf(C.Structure):
    _fields_ = [("kind", C.c_int), ("reserved", C.c_int), ("lam_star", C.c_double), ("delta1", C.c_double),
                ("delta2", C.c_double), ("mu_log10", C.c_double), ("sigma_log10", C.c_double),
                ("lam_min", C.c_double), ("lam_max", C.c_double)]


class agnvar_e13_opts(C.Structure):
    _fields_ = [("delta_threshold", C.c_double), ("d_delta_hist", C.c_void_p), ("d_sort_fallbacks", C.c_void_p),
                ("check_every", C.c_int32), ("reserved", C.c_int32)]


class agnvar_slice_opts(C.Structure):
    _fields_ = [("chains", C.c_int64), ("burn_in", C.c_int32), ("thin", C.c_int32), ("max_steps", C.c_int32),
                ("reserved", C.c_int32), ("width", C.c_double), ("d_density", C.c_void_p),
                ("density_points", C.c_int64), ("d_u_dbg", C.c_void_p)]


_lib = None


def lib():
    """Load libagnvar.so, compiling it with nvcc first when the sources changed since it was built (source hash,
    not mtimes).  Only a missing nvcc falls back to the shipped .so -- and then only if that .so was built from
    exactly these sources; a failed compilation raises."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    try:
        path = _build.build()
    except FileNotFoundError as exc:  # no nvcc on this machine
        if not _build.is_fresh():
            raise RuntimeError(f"libagnvar.so is missing or stale and nvcc is not available: {exc}") from exc
    L = C.CDLL(path)
    vp, i64, u64, u32, i32, dbl, sz = C.c_void_p, C.c_int64, C.c_uint64, C.c_uint32, C.c_int, C.c_double, C.c_size_t
    L.agnvar_workspace_bytes.restype = sz
    L.agnvar_workspace_bytes.argtypes = [i32, i64, i64, i32, i32, i64]
    L.agnvar_psd_bpl.restype = i32
    L.agnvar_psd_bpl.argtypes = [vp, i64, C.POINTER(agnvar_psd), vp, vp]
    L.agnvar_erdf_sample_sorted.restype = i32
    L.agnvar_erdf_sample_sorted.argtypes = [C.POINTER(agnvar_erdf), i64, i64, i64, i32, u64, u32, i32, vp, vp, vp,
                                            vp, sz, vp]
    L.agnvar_tk_generate.restype = i32
    L.agnvar_tk_generate.argtypes = [C.POINTER(agnvar_psd), i64, i64, i64, dbl, i32, i32, u64, u32, vp, vp, vp, sz,
                                     vp]
    L.agnvar_e13_iterate.restype = i32
    L.agnvar_e13_iterate.argtypes = [i64, i64, i32, vp, vp, vp, vp, i32, vp, vp, vp, C.POINTER(agnvar_e13_opts), vp, sz,
                                     vp]
    L.agnvar_slice_sample_sorted.restype = i32
    L.agnvar_slice_sample_sorted.argtypes = [C.POINTER(agnvar_erdf), i64, i64, i64, i32, u64, u32,
                                             C.POINTER(agnvar_slice_opts), vp, vp, vp, vp, sz, vp]
    L.agnvar_erdf_table.restype = i32
    L.agnvar_erdf_table.argtypes = [C.POINTER(agnvar_erdf), i64, i32, vp, vp]
    L.agnvar_periodogram.restype = i32
    L.agnvar_periodogram.argtypes = [i64, i64, i32, vp, dbl, i32, i32, C.POINTER(i64), vp, vp, vp, sz, vp]
    L.agnvar_structure_function.restype = i32
    L.agnvar_structure_function.argtypes = [i64, i64, i32, vp, C.POINTER(i64), i32, i32, vp, vp, vp, vp, vp, sz, vp]
    L.agnvar_static_scratch_bytes.restype = sz
    L.agnvar_static_scratch_bytes.argtypes = []
    L.agnvar_structure_function_static_bytes.restype = sz
    L.agnvar_structure_function_static_bytes.argtypes = [i64, i64, i32, i32]
    L.agnvar_structure_function_static.restype = i32
    L.agnvar_structure_function_static.argtypes = [i64, i64, i32, vp, C.POINTER(i64), i32, i32, vp, vp, vp, vp, vp]
    L.agnvar_delta_m_prob.restype = i32
    L.agnvar_delta_m_prob.argtypes = [i64, i64, i32, vp, C.POINTER(i64), i32, C.POINTER(dbl), i32, dbl, i32, dbl, vp, vp,
                                      vp, sz, vp]
    L.agnvar_ensemble_sf.restype = i32
    L.agnvar_ensemble_sf.argtypes = [i64, i64, i32, vp, i64, dbl, u64, u32, C.POINTER(i64), i32, i32, vp, vp, vp, vp, sz, vp]
    L.agnvar_moments.restype = i32
    L.agnvar_moments.argtypes = [i64, i64, i32, vp, vp, vp]
    L.agnvar_philox_u32.restype = i32
    L.agnvar_philox_u32.argtypes = [u64, u64, i64, u32, u32, vp, vp]
    L.agnvar_strerror.restype = C.c_char_p
    L.agnvar_strerror.argtypes = [i32]
    L.agnvar_version.restype = C.c_char_p
    L.agnvar_version.argtypes = []
    L.agnvar_launch_count.restype = u64
    L.agnvar_launch_count.argtypes = []
    L.agnvar_trace_begin.restype = i32
    L.agnvar_trace_begin.argtypes = []
    L.agnvar_trace_end.restype = i32
    L.agnvar_trace_end.argtypes = [i64, vp, vp, C.POINTER(i64)]
    L.agnvar_kernel_name.restype = C.c_char_p
    L.agnvar_kernel_name.argtypes = [i32]
    if _build.source_hash().encode() not in L.agnvar_version():
        raise RuntimeError("libagnvar.so does not match the sources in csrc/ (stale build)")
    _lib = L
    return L


def strerror(status):
    return lib().agnvar_strerror(int(status)).decode()


def version():
    return lib().agnvar_version().decode()


def launch_count():
    """Kernels launched by the library in this process so far."""
    return int(lib().agnvar_launch_count())


def trace_begin():
    _check(lib().agnvar_trace_begin(), "agnvar_trace_begin")


def trace_end(cap=1 << 20):
    """Returns a list of (kernel family name, device ms) in issue order for every launch since trace_begin()."""
    ids = (C.c_int32 * cap)()
    ms = (C.c_float * cap)()
    n = C.c_int64(0)
    _check(lib().agnvar_trace_end(cap, ids, ms, C.byref(n)), "agnvar_trace_end")
    m = min(int(n.value), cap)
    return [(lib().agnvar_kernel_name(ids[i]).decode(), float(ms[i])) for i in range(m)]


# ---- marshalling helpers --------------------------------------------------------------------------
def _dt(dtype):
    if dtype in (AGNVAR_F32, torch.float32, "f32", "float32"):
        return AGNVAR_F32, torch.float32
    if dtype in (AGNVAR_F64, torch.float64, "f64", "float64"):
        return AGNVAR_F64, torch.float64
    raise ValueError(f"dtype {dtype!r}: use float32 or float64")


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _on(device):
    """Make `device` current for the duration of a call: the library launches on the current device."""
    return torch.cuda.device(torch.device(device))


def _check(st, where):
    if st != 0:
        raise AgnvarError(st, where)


def _psd_array(psd):
    """psd: one (A, f_b, alpha_low, alpha_high) tuple/dict, a sequence of them, or an (array, count) pair already
    marshalled by this function (large batches: marshal once, reuse for every call)."""
    if isinstance(psd, tuple) and len(psd) == 2 and isinstance(psd[0], C.Array):
        return psd
    items = [psd] if isinstance(psd, (dict, tuple)) else list(psd)
    arr = (agnvar_psd * len(items))()
    for i, p in enumerate(items):
        if isinstance(p, dict):
            p = (p.get("A", 0.0), p["f_b"], p["alpha_low"], p["alpha_high"])
        arr[i] = agnvar_psd(float(p[0]), float(p[1]), float(p[2]), float(p[3]))
    return arr, len(items)


def _erdf_array(erdf):
    """erdf: one dict (kind, lam_star, delta1, delta2 | mu_log10, sigma_log10, lam_min, lam_max), a sequence of them,
    or an (array, count) pair already marshalled by this function."""
    if isinstance(erdf, tuple) and len(erdf) == 2 and isinstance(erdf[0], C.Array):
        return erdf
    items = [erdf] if isinstance(erdf, dict) else list(erdf)
    arr = (agnvar_erdf * len(items))()
    for i, e in enumerate(items):
        arr[i] = agnvar_erdf(int(e["kind"]), 0, float(e.get("lam_star", 1.0)), float(e.get("delta1", 0.0)),
                             float(e.get("delta2", 0.0)), float(e.get("mu_log10", 0.0)),
                             float(e.get("sigma_log10", 1.0)), float(e["lam_min"]), float(e["lam_max"]))
    return arr, len(items)


def marshal_params(cfg):
    """The C parameter arrays of a workload dict, built once and kept in it (65536 structs take tens of ms in Python)."""
    if "_c_params" not in cfg:
        cfg["_c_params"] = (_psd_array(cfg["psd"]), _erdf_array(cfg["erdf"]))
    return cfg["_c_params"]


_ws_cache = {}


def workspace_bytes(op, B, N, dtype, oversample=1, aux=0):
    return int(lib().agnvar_workspace_bytes(int(op), int(B), int(N), _dt(dtype)[0], int(oversample), int(aux)))


def workspace(nbytes, device=None):
    """A cached uint8 device tensor of at least nbytes (one per device; grown on demand)."""
    device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
    if device.index is None:
        device = torch.device("cuda", torch.cuda.current_device())
    cur = _ws_cache.get(device)
    if cur is None or cur.numel() < nbytes:
        _ws_cache[device] = None
        cur = torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device)
        _ws_cache[device] = cur
    return cur


def free_workspace():
    _ws_cache.clear()


# ---- the calls of include/agnvar.h ----------------------------------------------------------------
def agnvar_philox_u32(seed, i0, n, curve, tag, device="cuda"):
    """O1: raw Philox4x32-10 words [n][4] (int32 tensor holding the u32 bit patterns)."""
    with _on(device):
        out = torch.empty((n, 4), dtype=torch.int32, device=device)
        _check(lib().agnvar_philox_u32(int(seed), int(i0), int(n), int(curve), int(tag), _ptr(out), _stream()),
               "agnvar_philox_u32")
    return out


def agnvar_psd_bpl(f, psd, out=None):
    """S0: Eq. 3 at the fp64 device tensor f. psd = (A, f_b, alpha_low, alpha_high)."""
    arr, _ = _psd_array(psd)
    with _on(f.device):
        if out is None:
            out = torch.empty_like(f)
        _check(lib().agnvar_psd_bpl(_ptr(f), f.numel(), arr, _ptr(out), _stream()), "agnvar_psd_bpl")
    return out


def agnvar_erdf_table(erdf, grid_points=4096, device="cuda"):
    """S1's normalised cumulative table(s) C [n_erdf][grid_points] fp64 (O4)."""
    arr, n = _erdf_array(erdf)
    with _on(device):
        out = torch.empty((n, grid_points), dtype=torch.float64, device=device)
        _check(lib().agnvar_erdf_table(arr, n, int(grid_points), _ptr(out), _stream()), "agnvar_erdf_table")
    return out


def agnvar_erdf_sample_sorted(erdf, B, N, dtype, seed, curve0=0, grid_points=4096, want_perm0=True,
                              want_draw=False, device="cuda"):
    """S1: returns (sorted [B][N], perm0 [B][N] u32-as-int32 | None, draw [B][N] | None)."""
    code, tdt = _dt(dtype)
    arr, n = _erdf_array(erdf)
    with _on(device):
        srt = torch.empty((B, N), dtype=tdt, device=device)
        perm0 = torch.empty((B, N), dtype=torch.int32, device=device) if want_perm0 else None
        draw = torch.empty((B, N), dtype=tdt, device=device) if want_draw else None
        nb = workspace_bytes(OP_ERDF_SAMPLE_SORTED, B, N, code, 1, grid_points)
        ws = workspace(nb, srt.device)
        _check(lib().agnvar_erdf_sample_sorted(arr, n, B, N, code, int(seed), int(curve0), int(grid_points), _ptr(srt),
                                               _ptr(perm0), _ptr(draw), _ptr(ws), ws.numel(), _stream()),
               "agnvar_erdf_sample_sorted")
    return srt, perm0, draw


def agnvar_slice_sample_sorted(erdf, B, N, dtype, seed, chains, curve0=0, burn_in=50, thin=1, width=1.0, max_steps=8,
                               density=None, want_perm0=True, want_draw=False, want_u=False, device="cuda"):
    """NEXT-3: S1 by slice sampling (Neal 2003).  erdf kind 2 takes `density` [n_erdf][G] fp64 (device).
    Returns (sorted [B][N], perm0 | None, draw | None, u [B][N] fp64 | None)."""
    code, tdt = _dt(dtype)
    arr, n = _erdf_array(erdf)
    with _on(device):
        srt = torch.empty((B, N), dtype=tdt, device=device)
        perm0 = torch.empty((B, N), dtype=torch.int32, device=device) if want_perm0 else None
        draw = torch.empty((B, N), dtype=tdt, device=device) if want_draw else None
        u = torch.empty((B, N), dtype=torch.float64, device=device) if want_u else None
        if density is not None:
            assert density.dtype == torch.float64 and density.is_contiguous() and density.dim() == 2
        opts = agnvar_slice_opts(int(chains), int(burn_in), int(thin), int(max_steps), 0, float(width),
                                 density.data_ptr() if density is not None else None,
                                 int(density.shape[1]) if density is not None else 0,
                                 u.data_ptr() if u is not None else None)
        nb = workspace_bytes(OP_SLICE_SAMPLE_SORTED, B, N, code, 1, 0)
        ws = workspace(nb, srt.device)
        _check(lib().agnvar_slice_sample_sorted(arr, n, B, N, code, int(seed), int(curve0), C.byref(opts), _ptr(srt),
                                                _ptr(perm0), _ptr(draw), _ptr(ws), ws.numel(), _stream()),
               "agnvar_slice_sample_sorted")
    return srt, perm0, draw, u


def agnvar_tk_generate(psd, B, N, dt, oversample, dtype, seed, curve0=0, want_xnorm=True, want_anorm=True,
                       device="cuda"):
    """S2: returns (x_norm [B][N] | None, A_norm [B][N/2+1] | None)."""
    code, tdt = _dt(dtype)
    arr, n = _psd_array(psd)
    with _on(device):
        xn = torch.empty((B, N), dtype=tdt, device=device) if want_xnorm else None
        an = torch.empty((B, N // 2 + 1), dtype=tdt, device=device) if want_anorm else None
        nb = workspace_bytes(OP_TK_GENERATE, B, N, code, oversample, 0)
        ws = workspace(nb, (xn if xn is not None else an).device)
        _check(lib().agnvar_tk_generate(arr, n, B, N, float(dt), int(oversample), code, int(seed), int(curve0),
                                        _ptr(xn), _ptr(an), _ptr(ws), ws.numel(), _stream()), "agnvar_tk_generate")
    return xn, an


def agnvar_e13_iterate(anorm, sorted_vals, perm, max_iter, x=None, want_hist=False, want_xadj=False,
                       delta_threshold=0.0, want_delta=False, want_fallbacks=False, check_every=0):
    """L1-L6. perm is updated IN PLACE (in: idx_old of the first iteration, out: final permutation).
    delta_threshold > 0 adds the paper's stopping rule (Eq. 4); want_delta returns delta_k of every iteration.
    Returns dict(x, perm, iters_used, changed_hist | None, x_adj | None, delta_hist | None, sort_fallbacks | None)."""
    B, N = sorted_vals.shape
    code, tdt = _dt(sorted_vals.dtype)
    dev = sorted_vals.device
    assert anorm.dtype == tdt and anorm.shape == (B, N // 2 + 1) and anorm.is_contiguous()
    assert perm.dtype == torch.int32 and perm.shape == (B, N) and perm.is_contiguous() and sorted_vals.is_contiguous()
    with _on(dev):
        if x is None:
            x = torch.empty((B, N), dtype=tdt, device=dev)
        iters = torch.empty((B,), dtype=torch.int32, device=dev)
        hist = torch.empty((B, max_iter), dtype=torch.int64, device=dev) if want_hist else None
        xadj = torch.empty((B, N), dtype=tdt, device=dev) if want_xadj else None
        dhist = torch.empty((B, max_iter), dtype=torch.float64, device=dev) if want_delta else None
        fb = torch.empty((B,), dtype=torch.int32, device=dev) if want_fallbacks else None
        delta_mode = want_delta or delta_threshold > 0.0
        opts = agnvar_e13_opts(float(delta_threshold), dhist.data_ptr() if dhist is not None else None,
                               fb.data_ptr() if fb is not None else None, int(check_every), 0)
        nb = workspace_bytes(OP_E13_ITERATE, B, N, code, 1, 1 if delta_mode else 0)
        ws = workspace(nb, dev)
        _check(lib().agnvar_e13_iterate(B, N, code, _ptr(anorm), _ptr(sorted_vals), _ptr(perm), _ptr(x), int(max_iter),
                                        _ptr(iters), _ptr(hist), _ptr(xadj), C.byref(opts), _ptr(ws), ws.numel(),
                                        _stream()), "agnvar_e13_iterate")
    return {"x": x, "perm": perm, "iters_used": iters, "changed_hist": hist, "x_adj": xadj, "delta_hist": dhist,
            "sort_fallbacks": fb}


def agnvar_periodogram(x, dt, norm=0, bin_edges=None):
    """P: x [B][N] -> P [B][N/2] fp64, or (Pbin [B][nbins] fp64, counts [nbins] i64) with integer bin edges."""
    B, N = x.shape
    code, _ = _dt(x.dtype)
    dev = x.device
    nbins = 0 if bin_edges is None else len(bin_edges) - 1
    with _on(dev):
        out = torch.empty((B, nbins if nbins else N // 2), dtype=torch.float64, device=dev)
        counts = torch.empty((nbins,), dtype=torch.int64, device=dev) if nbins else None
        edges = (C.c_int64 * (nbins + 1))(*[int(e) for e in bin_edges]) if nbins else None
        nb = workspace_bytes(OP_PERIODOGRAM, B, N, code, 1, nbins)
        ws = workspace(nb, dev)
        _check(lib().agnvar_periodogram(B, N, code, _ptr(x), float(dt), int(norm), nbins, edges, _ptr(out), _ptr(counts),
                                        _ptr(ws), ws.numel(), _stream()), "agnvar_periodogram")
    return out if not nbins else (out, counts)


def agnvar_structure_function(x, lags, mag=False, want_rep=False):
    """NEXT-2 (Eq. A6): x [B][N] -> dict(sf2 [B][nlags] fp64, pairs [nlags] i64, rep_mean / rep_stderr [nlags] | None)."""
    B, N = x.shape
    code, _ = _dt(x.dtype)
    dev = x.device
    nl = len(lags)
    arr = (C.c_int64 * nl)(*[int(l) for l in lags])
    with _on(dev):
        sf2 = torch.empty((B, nl), dtype=torch.float64, device=dev)
        pairs = torch.empty((nl,), dtype=torch.int64, device=dev)
        mean = torch.empty((nl,), dtype=torch.float64, device=dev) if want_rep else None
        se = torch.empty((nl,), dtype=torch.float64, device=dev) if want_rep else None
        ws = workspace(workspace_bytes(OP_STRUCTURE_FUNCTION, B, N, code, 1, nl), dev)
        _check(lib().agnvar_structure_function(B, N, code, _ptr(x), arr, nl, 1 if mag else 0, _ptr(sf2), _ptr(pairs),
                                               _ptr(mean), _ptr(se), _ptr(ws), ws.numel(), _stream()),
               "agnvar_structure_function")
    return {"sf2": sf2, "pairs": pairs, "rep_mean": mean, "rep_stderr": se}


AGNVAR_ESTATIC_LIMIT = 5


def agnvar_structure_function_static(x, lags, mag=False, want_rep=False, out=None):
    """agnvar_structure_function for a caller that has no scratch memory to offer (include/agnvar.h, "SF without a
    workspace").

    Use it where device allocation is not an option -- a plug-in that only receives tensors, a process whose device
    memory already belongs to somebody else's pool, a loop that cannot afford the stall an allocation may cause.  The
    library then works in an 8 MiB array that is part of libagnvar.so (every GPU that loads the library holds it until
    the process exits); this call allocates nothing on the device when `out` is given.

    x [B][N] float32 / float64 on the GPU; at most 256 lags; the request must fit the array
    (static_scratch_need(...) <= static_scratch_bytes(), e.g. 64 curves x 2^20 samples x 64 lags without magnitudes,
    about 10^6 samples in total with mag=True) or AgnvarError(status AGNVAR_ESTATIC_LIMIT) is raised and nothing runs.
    out: the dict a previous call returned (its tensors are overwritten), so that a caller that may not allocate can
    create the outputs once at start-up; None lets torch allocate them.
    Make the first call on each device at start-up (it looks up the array's device address).  All calls on a device
    share the one array: keep them on one stream, or order them with events; calls that overlap on the GPU corrupt
    each other's sums.  Results are identical to agnvar_structure_function's (same kernels)."""
    B, N = x.shape
    code, _ = _dt(x.dtype)
    dev = x.device
    nl = len(lags)
    arr = (C.c_int64 * nl)(*[int(l) for l in lags])
    with _on(dev):
        if out is None:
            out = {"sf2": torch.empty((B, nl), dtype=torch.float64, device=dev),
                   "pairs": torch.empty((nl,), dtype=torch.int64, device=dev),
                   "rep_mean": torch.empty((nl,), dtype=torch.float64, device=dev) if want_rep else None,
                   "rep_stderr": torch.empty((nl,), dtype=torch.float64, device=dev) if want_rep else None}
        elif tuple(out["sf2"].shape) != (B, nl) or out["pairs"].numel() != nl:
            raise ValueError("out does not have the shapes of this request")
        _check(lib().agnvar_structure_function_static(B, N, code, _ptr(x), arr, nl, 1 if mag else 0, _ptr(out["sf2"]),
                                                      _ptr(out["pairs"]), _ptr(out["rep_mean"]), _ptr(out["rep_stderr"]),
                                                      _stream()),
               "agnvar_structure_function_static")
    return out


def static_scratch_bytes():
    """Size of the array agnvar_structure_function_static works in (bytes held on every GPU that loads the library)."""
    return int(lib().agnvar_static_scratch_bytes())


def static_scratch_need(B, N, nlags, mag=False):
    """Bytes of that array a request would use (0 for invalid arguments); it runs iff this is <= static_scratch_bytes()."""
    return int(lib().agnvar_structure_function_static_bytes(int(B), int(N), int(nlags), 1 if mag else 0))


def agnvar_delta_m_prob(x, lags, dm_ref, m_zero=0.0, m_cut=None):
    """NEXT-2: x [B][N] -> (prob [B][nlags][nref] fp64, considered [B][nlags] i64)."""
    B, N = x.shape
    code, _ = _dt(x.dtype)
    dev = x.device
    nl, nr = len(lags), len(dm_ref)
    larr = (C.c_int64 * nl)(*[int(l) for l in lags])
    rarr = (C.c_double * nr)(*[float(r) for r in dm_ref])
    with _on(dev):
        prob = torch.empty((B, nl, nr), dtype=torch.float64, device=dev)
        cons = torch.empty((B, nl), dtype=torch.int64, device=dev)
        ws = workspace(workspace_bytes(OP_DELTA_M_PROB, B, N, code, 1, nl), dev)
        _check(lib().agnvar_delta_m_prob(B, N, code, _ptr(x), larr, nl, rarr, nr, float(m_zero), 0 if m_cut is None else 1,
                                         0.0 if m_cut is None else float(m_cut), _ptr(prob), _ptr(cons), _ptr(ws),
                                         ws.numel(), _stream()), "agnvar_delta_m_prob")
    return prob, cons


def agnvar_ensemble_sf(x, n_sub, keep, seed, lags, curve0=0, mag=False):
    """NEXT-4 (Fig. 7-8): ensemble SF over masked consecutive sub-samples of every curve.
    Returns dict(sf2 [nlags] fp64, pairs [nlags] i64, offsets [B] i64)."""
    B, N = x.shape
    code, _ = _dt(x.dtype)
    dev = x.device
    nl = len(lags)
    arr = (C.c_int64 * nl)(*[int(l) for l in lags])
    with _on(dev):
        sf2 = torch.empty((nl,), dtype=torch.float64, device=dev)
        pairs = torch.empty((nl,), dtype=torch.int64, device=dev)
        offs = torch.empty((B,), dtype=torch.int64, device=dev)
        ws = workspace(workspace_bytes(OP_ENSEMBLE_SF, B, n_sub, code, 1, nl), dev)
        _check(lib().agnvar_ensemble_sf(B, N, code, _ptr(x), int(n_sub), float(keep), int(seed), int(curve0), arr, nl,
                                        1 if mag else 0, _ptr(sf2), _ptr(pairs), _ptr(offs), _ptr(ws), ws.numel(), _stream()),
               "agnvar_ensemble_sf")
    return {"sf2": sf2, "pairs": pairs, "offsets": offs}


def agnvar_moments(x):
    """Per-curve mean, variance, skewness, excess kurtosis: [B][4] fp64 (Fig. 2's check of the TK95 output PDF)."""
    B, N = x.shape
    code, _ = _dt(x.dtype)
    with _on(x.device):
        out = torch.empty((B, 4), dtype=torch.float64, device=x.device)
        _check(lib().agnvar_moments(B, N, code, _ptr(x), _ptr(out), _stream()), "agnvar_moments")
    return out

"""ctypes front end of the CPU oracle (oracle/agnvar_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference leg may import this package.  It shares nothing with the CUDA
path (paper_1909_06374_b200/): argument marshalling to numpy arrays only; every number is
computed by the C++ file, whose functions cite the passage of PAPER.md they follow.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None

_f64p = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_u32p = np.ctypeslib.ndpointer(dtype=np.uint32, flags="C_CONTIGUOUS")
_i64p = np.ctypeslib.ndpointer(dtype=np.int64, flags="C_CONTIGUOUS")


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        _lib = C.CDLL(path)
        _lib.orc_u53.restype = C.c_double
        _lib.orc_u53.argtypes = [C.c_uint32, C.c_uint32]
        _lib.orc_psd_unit_variance_A.restype = C.c_double
        _lib.orc_psd_unit_variance_A.argtypes = [C.c_int64, C.c_double, C.c_double, C.c_double, C.c_double]
        _lib.orc_delta_rms.restype = C.c_double
        _lib.orc_delta_rms.argtypes = [C.c_void_p, C.c_void_p, C.c_int64]
    return _lib


def _d(x):
    return np.ascontiguousarray(x, dtype=np.float64)


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


# ---- O1 Philox ---------------------------------------------------------------------------------
def philox4x32_10(ctr, key):
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def philox_stream(seed, i, b, tag):
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox_stream(C.c_uint64(seed), C.c_uint64(i), C.c_uint32(b), C.c_uint32(tag), _p(out))
    return out


def u53(wa, wb):
    return lib().orc_u53(int(wa), int(wb))


def tk_normal_pair(seed, j, b):
    gr, gi = C.c_double(), C.c_double()
    lib().orc_tk_normal_pair(C.c_uint64(seed), C.c_uint64(j), C.c_uint32(b), C.byref(gr), C.byref(gi))
    return gr.value, gi.value


# ---- DFT / FFT ---------------------------------------------------------------------------------
def _cplx_call(fn, x, sign):
    x = np.asarray(x)
    re = _d(x.real)
    im = _d(x.imag) if np.iscomplexobj(x) else None
    n = re.shape[0]
    ore, oim = np.empty(n), np.empty(n)
    fn(_p(re), _p(im), C.c_int64(n), C.c_int(sign), _p(ore), _p(oim))
    return ore + 1j * oim


def dft_naive(x, sign=-1):
    return _cplx_call(lib().orc_dft_naive, x, sign)


def fft(x, sign=-1):
    """Always the recursive FFT (pin target: compare with dft_naive)."""
    return _cplx_call(lib().orc_fft, x, sign)


def rfft(x):
    x = _d(x)
    n = x.shape[0]
    re, im = np.empty(n // 2 + 1), np.empty(n // 2 + 1)
    lib().orc_rfft(_p(x), C.c_int64(n), _p(re), _p(im))
    return re + 1j * im


def irfft(X, n):
    X = np.asarray(X, dtype=np.complex128)
    re, im = _d(X.real), _d(X.imag)
    out = np.empty(n)
    lib().orc_irfft(_p(re), _p(im), C.c_int64(n), _p(out))
    return out


# ---- O2 PSD ------------------------------------------------------------------------------------
def psd_bpl(f, A, f_b, a_lo, a_hi):
    f = _d(f)
    out = np.empty_like(f)
    lib().orc_psd_bpl(_p(f), C.c_int64(f.size), C.c_double(A), C.c_double(f_b), C.c_double(a_lo),
                      C.c_double(a_hi), _p(out))
    return out


def psd_unit_variance_A(M, dt, f_b, a_lo, a_hi):
    return lib().orc_psd_unit_variance_A(int(M), float(dt), float(f_b), float(a_lo), float(a_hi))


# ---- O3 TK95 -----------------------------------------------------------------------------------
def tk_generate(A, f_b, a_lo, a_hi, N, dt, oversample, seed, b, want_full=False):
    M = N * oversample
    Xre = np.empty(M // 2 + 1) if want_full else None
    Xim = np.empty(M // 2 + 1) if want_full else None
    xf = np.empty(M) if want_full else None
    xn = np.empty(N)
    An = np.empty(N // 2 + 1)
    rc = lib().orc_tk_generate(C.c_double(A), C.c_double(f_b), C.c_double(a_lo), C.c_double(a_hi),
                               C.c_int64(N), C.c_double(dt), C.c_int(oversample), C.c_uint64(seed),
                               C.c_uint32(b), _p(Xre), _p(Xim), _p(xf), _p(xn), _p(An))
    if rc != 0:
        raise ValueError("orc_tk_generate: bad arguments")
    out = {"x_norm": xn, "A_norm": An}
    if want_full:
        out.update({"X": Xre + 1j * Xim, "x_full": xf})
    return out


# ---- O4 ERDF -----------------------------------------------------------------------------------
def _erdf_args(e):
    return [C.c_int(int(e["kind"])), C.c_double(e.get("lam_star", 1.0)), C.c_double(e.get("delta1", 0.0)),
            C.c_double(e.get("delta2", 0.0)), C.c_double(e.get("mu_log10", 0.0)),
            C.c_double(e.get("sigma_log10", 1.0)), C.c_double(e["lam_min"]), C.c_double(e["lam_max"])]


def erdf_table(erdf, G):
    u, p, Cc = np.empty(G), np.empty(G), np.empty(G)
    lib().orc_erdf_table(*_erdf_args(erdf), C.c_int64(G), _p(u), _p(p), _p(Cc))
    return u, p, Cc


def erdf_draw(erdf, G, N, seed, b, dtype):
    """dtype 0: fp32-rounded values, 1: fp64.  Returns (lambda in draw order, the uniforms used)."""
    lam, U = np.empty(N), np.empty(N)
    lib().orc_erdf_draw(*_erdf_args(erdf), C.c_int64(G), C.c_int64(N), C.c_uint64(seed), C.c_uint32(b),
                        C.c_int(dtype), _p(lam), _p(U))
    return lam, U


# ---- sorting -----------------------------------------------------------------------------------
def stable_argsort(x):
    x = _d(x)
    idx = np.empty(x.size, dtype=np.uint32)
    lib().orc_stable_argsort(_p(x), C.c_int64(x.size), _p(idx))
    return idx


def rank_bruteforce(x):
    x = _d(x)
    r = np.empty(x.size, dtype=np.uint32)
    lib().orc_rank_bruteforce(_p(x), C.c_int64(x.size), _p(r))
    return r


def erdf_sample_sorted(erdf, G, N, seed, b, dtype):
    """O4 + Q15: the draw, its stable ascending sort and perm0 (time index of the r-th smallest)."""
    lam, _ = erdf_draw(erdf, G, N, seed, b, dtype)
    perm0 = stable_argsort(lam)
    return lam[perm0].copy(), perm0, lam


# ---- O6 E13 ------------------------------------------------------------------------------------
def e13_step(A_norm, sorted_vals, idx_old, x_sim):
    A_norm, sorted_vals, x_sim = _d(A_norm), _d(sorted_vals), _d(x_sim)
    idx_old = np.ascontiguousarray(idx_old, dtype=np.uint32)
    n = x_sim.size
    x_adj, x_next = np.empty(n), np.empty(n)
    idx_new = np.empty(n, dtype=np.uint32)
    ch = C.c_int64(0)
    lib().orc_e13_step(C.c_int64(n), _p(A_norm), _p(sorted_vals), _p(idx_old), _p(x_sim), _p(x_adj),
                       _p(idx_new), _p(x_next), C.byref(ch))
    return x_adj, idx_new, x_next, ch.value


def e13_iterate(A_norm, sorted_vals, perm0, max_iter):
    A_norm, sorted_vals = _d(A_norm), _d(sorted_vals)
    perm = np.array(perm0, dtype=np.uint32, copy=True)
    n = sorted_vals.size
    x, x_adj = np.empty(n), np.empty(n)
    iters = C.c_int32(0)
    hist = np.zeros(max_iter, dtype=np.int64)
    rc = lib().orc_e13_iterate(C.c_int64(n), _p(A_norm), _p(sorted_vals), _p(perm), _p(x), C.c_int(max_iter),
                               C.byref(iters), _p(hist), _p(x_adj))
    if rc != 0:
        raise ValueError("orc_e13_iterate: bad arguments")
    return {"x": x, "perm": perm, "iters_used": iters.value, "changed_hist": hist, "x_adj_last": x_adj}


# ---- O7 periodogram ----------------------------------------------------------------------------
def periodogram(x, dt, norm):
    x = _d(x)
    P = np.empty(x.size // 2)
    lib().orc_periodogram(_p(x), C.c_int64(x.size), C.c_double(dt), C.c_int(norm), _p(P))
    return P


def periodogram_binned(x, dt, norm, edges):
    x = _d(x)
    edges = np.ascontiguousarray(edges, dtype=np.int64)
    nb = edges.size - 1
    out = np.empty(nb)
    cnt = np.empty(nb, dtype=np.int64)
    lib().orc_periodogram_binned(_p(x), C.c_int64(x.size), C.c_double(dt), C.c_int(norm), C.c_int(nb),
                                 _p(edges), _p(out), _p(cnt))
    return out, cnt


# ---- NEXT-1: delta_i (Eq. 4) ---------------------------------------------------------------------
def delta_rms(x_new, x_old):
    x_new, x_old = _d(x_new), _d(x_old)
    return lib().orc_delta_rms(_p(x_new), _p(x_old), x_new.size)


def e13_iterate_delta(A_norm, sorted_vals, perm0, max_iter, threshold=0.0):
    A_norm, sorted_vals = _d(A_norm), _d(sorted_vals)
    perm = np.array(perm0, dtype=np.uint32, copy=True)
    n = sorted_vals.size
    x = np.empty(n)
    iters = C.c_int32(0)
    hist = np.zeros(max_iter, dtype=np.int64)
    dhist = np.zeros(max_iter)
    rc = lib().orc_e13_iterate_delta(C.c_int64(n), _p(A_norm), _p(sorted_vals), _p(perm), _p(x), C.c_int(max_iter),
                                     C.c_double(threshold), C.byref(iters), _p(hist), _p(dhist))
    if rc != 0:
        raise ValueError("orc_e13_iterate_delta: bad arguments")
    return {"x": x, "perm": perm, "iters_used": iters.value, "changed_hist": hist, "delta_hist": dhist}


# ---- NEXT-2: structure function (Eq. A6), representative SF (Eq. 6), P(|dm| > dm_ref | tau) ---------
def structure_function(x, lags, mag=False):
    x = _d(x)
    lags = np.ascontiguousarray(lags, dtype=np.int64)
    sf2 = np.empty(lags.size)
    pairs = np.empty(lags.size, dtype=np.int64)
    lib().orc_structure_function(_p(x), C.c_int64(x.size), _p(lags), C.c_int(lags.size), C.c_int(1 if mag else 0),
                                 _p(sf2), _p(pairs))
    return sf2, pairs


def sf_representative(sf2):
    sf2 = _d(sf2)
    nsim, nl = sf2.shape
    mean, se = np.empty(nl), np.empty(nl)
    lib().orc_sf_representative(_p(sf2), C.c_int(nsim), C.c_int(nl), _p(mean), _p(se))
    return mean, se


def delta_m_prob(x, lags, dm_ref, m_zero=0.0, m_cut=None):
    x = _d(x)
    lags = np.ascontiguousarray(lags, dtype=np.int64)
    dm_ref = _d(dm_ref)
    prob = np.empty((lags.size, dm_ref.size))
    cons = np.empty(lags.size, dtype=np.int64)
    lib().orc_delta_m_prob(_p(x), C.c_int64(x.size), _p(lags), C.c_int(lags.size), _p(dm_ref), C.c_int(dm_ref.size),
                           C.c_double(m_zero), C.c_int(0 if m_cut is None else 1),
                           C.c_double(0.0 if m_cut is None else m_cut), _p(prob), _p(cons))
    return prob, cons


# ---- NEXT-4: ensemble SF of masked sub-segments (Fig. 7-8), output-PDF moments (Fig. 2) -----------------
def ensemble_sf(x, n_sub, keep, seed, curve0, lags, mag=False):
    x = np.ascontiguousarray(x, dtype=np.float64)
    B, N = x.shape
    lags = np.ascontiguousarray(lags, dtype=np.int64)
    sf2 = np.empty(lags.size)
    pairs = np.empty(lags.size, dtype=np.int64)
    offs = np.empty(B, dtype=np.int64)
    lib().orc_ensemble_sf(_p(x), C.c_int64(B), C.c_int64(N), C.c_int64(n_sub), C.c_double(keep), C.c_uint64(seed),
                          C.c_uint32(curve0), _p(lags), C.c_int(lags.size), C.c_int(1 if mag else 0), _p(sf2), _p(pairs),
                          _p(offs))
    return sf2, pairs, offs


def moments(x):
    x = _d(x)
    out = np.empty(4)
    lib().orc_moments(_p(x), C.c_int64(x.size), _p(out))
    return out


# ---- NEXT-3: slice sampling (Neal 2003) -----------------------------------------
def slice_sample(erdf, N, chains, seed, b, dtype, burn_in=50, thin=1, w=1.0, m=8, table=None):
    """erdf: dict as for erdf_draw (kind 0 / 1), or kind 2 with `table` = un-normalised density on a uniform grid
    over [log10 lam_min, log10 lam_max].  Returns (lambda [N] in draw order, u = log10 lambda before rounding)."""
    lam, u = np.empty(N), np.empty(N)
    tab = _d(table) if table is not None else None
    G = len(tab) if tab is not None else 0
    assert N % chains == 0
    lib().orc_slice_sample(*_erdf_args(erdf), _p(tab) if tab is not None else None, C.c_int64(G), C.c_int64(N),
                           C.c_int64(chains), C.c_int(burn_in), C.c_int(thin), C.c_double(w), C.c_int(m),
                           C.c_uint64(seed), C.c_uint32(b), C.c_int(dtype), _p(lam), _p(u))
    return lam, u

"""One pass of the whole hot path (S1, S2, L1-L6, P) for one batch of curves.

Pure sequencing of the C-ABI calls; no arithmetic of the method happens here.
"""
import torch

from . import binding as _b
from . import workloads as _w


def generate_light_curves(cfg, device="cuda", host_out=None, want_hist=False, curve0=0, want_fallbacks=False,
                          delta_threshold=0.0, want_delta=False, phase_hook=None):
    """Run erdf_sample_sorted -> tk_generate -> e13_iterate (-> periodogram if cfg['nbins']) for cfg
    (a dict from workloads.config).  Returns dict(x, perm, iters_used, changed_hist, pbin, counts).

    host_out: optional pinned host tensor [B][N]; when given, the final light curves are copied into it
    (device -> host) on the current stream and the call synchronises, so that the result is usable on
    return -- this is the end-to-end entry point timed by bench.py's e2e leg.
    phase_hook: optional callable(name), called before each C-ABI call ("S1", "S2", "E13", "P") and at the end ("end");
    bench.py uses it to attribute traced launches to the call that made them.
    """
    hook = phase_hook if phase_hook is not None else (lambda name: None)
    B, N = cfg["B"], cfg["N"]
    psd_c, erdf_c = _b.marshal_params(cfg)
    hook("S1")
    if cfg.get("sampler", "inverse_cdf") == "slice":
        # the paper's own sampler for the random draw (NEXT-3): cfg["slice"] = dict(chains, burn_in, thin,
        # width, max_steps); same distribution as the inverse-CDF sampler, different samples
        so = dict(chains=min(N, 4096), burn_in=50, thin=1, width=1.0, max_steps=8)
        so.update(cfg.get("slice", {}))
        srt, perm, _, _ = _b.agnvar_slice_sample_sorted(erdf_c, B, N, cfg["dtype"], cfg["seed"], curve0=curve0,
                                                        device=device, **so)
    else:
        srt, perm, _ = _b.agnvar_erdf_sample_sorted(erdf_c, B, N, cfg["dtype"], cfg["seed"], curve0,
                                                    cfg["grid_points"], device=device)
    hook("S2")
    _, anorm = _b.agnvar_tk_generate(psd_c, B, N, cfg["dt"], cfg["oversample"], cfg["dtype"], cfg["seed"],
                                     curve0, want_xnorm=False, device=device)
    hook("E13")
    out = _b.agnvar_e13_iterate(anorm, srt, perm, cfg["max_iter"], want_hist=want_hist, want_fallbacks=want_fallbacks,
                                delta_threshold=delta_threshold, want_delta=want_delta)
    out["pbin"] = out["counts"] = None
    if cfg.get("nbins", 0):
        hook("P")
        out["pbin"], out["counts"] = _b.agnvar_periodogram(out["x"], cfg["dt"], 0,
                                                           _w.log_bin_edges(N, cfg["nbins"]))
    hook("end")
    if host_out is not None:
        host_out.copy_(out["x"], non_blocking=True)
        out["iters_host"] = out["iters_used"].cpu()  # synchronises the stream
        out["x_host"] = host_out
    return out

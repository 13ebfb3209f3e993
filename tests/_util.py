"""Shared helpers of the parity tests: seeded problems, the GPU chain through the C ABI, error measure."""
from __future__ import annotations

import numpy as np

from paper_2106_04649_b200 import configs, gen


def rel_l2(x, ref):
    x = np.asarray(x, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    den = np.linalg.norm(ref)
    return float(np.linalg.norm(x - ref) / den) if den > 0 else float(np.linalg.norm(x))


def problem(cfg, focs=None):
    """(R [n][n][nt], Gd [nfoc][n][nt], td [nfoc][n]) fp32 from the seeded generator."""
    base = gen.base_traces(cfg)
    R = gen.R_full(cfg, base)
    Gd, td = gen.first_arrivals(cfg, focs=focs)
    return R, Gd, td


def gpu_chain(cfg, R, Gd, td, niter=None, regime=0, keep_iters=True, host_api=False, outputs=("f1plus", "f1min", "G", "Gplus", "Gminus"),
              fft_path=0, streamed=None, rhat_format=0, rhat_layout=0):
    """Runs the CUDA path through the C ABI; returns numpy arrays like oracle.marchenko does.
    streamed = (resident_rows, window_rows): out-of-core R^ (mk_create_streamed); rhat_format: MK_OPT_RHAT_FORMAT; rhat_layout: MK_OPT_RHAT_LAYOUT."""
    import torch
    from paper_2106_04649_b200 import binding as B
    niter = cfg.niter if niter is None else niter
    nfoc = Gd.shape[0]
    dev = torch.device("cuda:0")
    out = {}
    with B.Marchenko(cfg.n, cfg.n, cfg.nt, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax, streamed=streamed) as mk:
        mk.set_option(B.MK_OPT_EPS_SAMPLES, cfg.eps)
        mk.set_option(B.MK_OPT_REGIME, regime)
        mk.set_option(B.MK_OPT_FFT_PATH, fft_path)
        mk.set_option(B.MK_OPT_RHAT_FORMAT, rhat_format)
        mk.set_option(B.MK_OPT_RHAT_LAYOUT, rhat_layout)
        if host_api:
            mk.load_R_host(np.ascontiguousarray(R))
            houts = {nm: np.empty((nfoc, cfg.n, cfg.nt), np.float32) for nm in outputs + ("N_last",)}
            mk.run_host(np.ascontiguousarray(Gd), np.ascontiguousarray(td), niter, houts)
            out.update(houts)
            out["regime_used"] = int(mk.get_info(B.MK_INFO_REGIME_USED))
            return out
        # ingest in two uneven chunks to exercise shot0 / nshots
        cut = max(1, (2 * cfg.n) // 3)
        if rhat_format:   # compressed R^ is ingested in whole 16-shot blocks
            cut = max(16, cut // 16 * 16) if cfg.n > 16 else cfg.n
        mk.load_R(torch.from_numpy(np.ascontiguousarray(R[:cut])).to(dev), 0)
        if cut < cfg.n:
            mk.load_R(torch.from_numpy(np.ascontiguousarray(R[cut:])).to(dev), cut)
        dGd = torch.from_numpy(np.ascontiguousarray(Gd)).to(dev)
        dtd = torch.from_numpy(np.ascontiguousarray(td)).to(dev)
        if keep_iters:
            mk.begin(dGd, dtd)
            its = []
            buf = torch.empty((nfoc, cfg.n, cfg.nt), dtype=torch.float32, device=dev)
            for _ in range(niter):
                mk.step(buf)
                its.append(buf.cpu().numpy().copy())
            out["N_iters"] = np.stack(its)
            douts = {nm: torch.empty((nfoc, cfg.n, cfg.nt), dtype=torch.float32, device=dev) for nm in outputs}
            mk.finish(douts)
        else:
            douts = {nm: torch.empty((nfoc, cfg.n, cfg.nt), dtype=torch.float32, device=dev) for nm in outputs + ("N_last",)}
            mk.run(dGd, dtd, niter, douts)
        torch.cuda.synchronize()
        for nm, t in douts.items():
            out[nm] = t.cpu().numpy()
        out["regime_used"] = int(mk.get_info(B.MK_INFO_REGIME_USED))
        out["h2d_bytes"] = mk.get_info(B.MK_INFO_H2D_BYTES)
        out["rhat_bytes_padded"] = mk.get_info(B.MK_INFO_RHAT_BYTES_PADDED)
    return out


def calibrated(cfg, target=0.5, iters=4):
    """Reduced copies of a config need their own amplitude constant: scale A_R (a power of two, so the generator's
    traces scale exactly) until the oracle's ||N_i|| / ||N_{i-1}|| is about `target` after `iters` steps."""
    import oracle
    from dataclasses import replace
    R, Gd, td = problem(cfg, focs=[cfg.nfoc // 2])
    o = oracle.marchenko(R, Gd, td, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax, iters, cfg.eps, want=())
    nrm = [np.linalg.norm(o["N_iters"][i]) for i in range(iters)]
    ratio = nrm[-1] / max(nrm[-2], 1e-300)
    scale = 2.0 ** np.round(np.log2(target / ratio)) if ratio > 0 else 1.0
    return replace(cfg, A_R=cfg.A_R * float(scale))

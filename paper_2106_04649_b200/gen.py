"""Seeded synthetic input generator (SURVEY.md §8(d) "Generator contract").

Serves BOTH the CUDA path and the oracle with identical bytes.  It holds none of the method's
arithmetic: no convolution, no Fourier transform, no window, no Neumann step — only the recipe that
makes the inputs R (reflection response), G_d (first arrivals) and t_d (their traveltimes):

* a counter-based RNG (splitmix64 finaliser over seed/stream/index), so every trace is a pure
  function of (config, s, r) and any chunk or subset can be regenerated without storing R;
* a laterally invariant layer model -> hyperbolic moveouts of primaries and first-order internal
  multiples, each carrying a zero-phase Ricker wavelet evaluated analytically (exact fractional
  shift) and set to exactly zero for |u| > cfg.half_support, so R is causal and confined to
  [0, nt/2);
* optional per-trace white Gaussian noise (config 3) on samples [0, nt/2);
* G_d = Ricker(t - t_d) with the straight-ray traveltime t_d through the top-layer velocity.

The inputs stand in for the paper's "oneD" data sets, which are not available.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

from .configs import Config

_U64 = np.uint64
_GOLD = _U64(0x9E3779B97F4A7C15)
_M1 = _U64(0xBF58476D1CE4E5B9)
_M2 = _U64(0x94D049BB133111EB)
_STREAM_MUL = _U64(0xD1B54A32D192ED03)

# RNG streams
_S_DT, _S_V, _S_R, _S_SIGN, _S_NOISE = 1, 2, 3, 4, 5


def _mix(x: np.ndarray) -> np.ndarray:
    """splitmix64 output function (Steele, Lea & Flood 2014) on uint64 arrays (wrapping arithmetic)."""
    with np.errstate(over="ignore"):
        z = x + _GOLD
        z = (z ^ (z >> _U64(30))) * _M1
        z = (z ^ (z >> _U64(27))) * _M2
        return z ^ (z >> _U64(31))


def _key(seed: int, stream: int) -> np.uint64:
    with np.errstate(over="ignore"):
        return _mix(np.asarray(_U64(seed) ^ (_U64(stream) * _STREAM_MUL), dtype=_U64))[()]


def uniforms(seed: int, stream: int, idx) -> np.ndarray:
    """U[0,1) doubles from the top 53 bits; a pure function of (seed, stream, idx)."""
    idx = np.asarray(idx, dtype=_U64)
    with np.errstate(over="ignore"):
        z = _mix(_key(seed, stream) + idx * _GOLD)
    return (z >> _U64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


# ----------------------------------------------------------------------------------------------
# layer model
# ----------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class LayerModel:
    t0: np.ndarray      # [L] two-way zero-offset time to interface l
    V: np.ndarray       # [L] sum_j<=l v_j^2 dt_j
    v: np.ndarray       # [L] interval velocities (v[0] = top layer)
    r: np.ndarray       # [L] reflection coefficients


def layer_model(cfg: Config) -> LayerModel:
    L = cfg.nlayers
    i = np.arange(L)
    seed = cfg.rseed
    dts = (0.6 + 0.8 * uniforms(seed, _S_DT, i)) * 0.30 * cfg.nt * cfg.dt / L
    v = 1500.0 + 1500.0 * uniforms(seed, _S_V, i)
    u = uniforms(seed, _S_R, i)
    if cfg.refl == "uniform03":
        r = -0.3 + 0.6 * u
    elif cfg.refl == "randsign025":
        sign = np.where(uniforms(seed, _S_SIGN, i) < 0.5, -1.0, 1.0)
        r = sign * (0.05 + 0.20 * u)
    else:
        raise ValueError(cfg.refl)
    t0 = np.cumsum(dts)
    V = np.cumsum(v * v * dts)
    return LayerModel(t0=t0, V=V, v=v, r=r)


def _events(model: LayerModel):
    """(t0, vrms^2, amplitude) of every primary and first-order internal multiple."""
    L = len(model.t0)
    t0s, v2s, amps = [], [], []
    trans = 1.0
    for l in range(L):
        t0s.append(model.t0[l])
        v2s.append(model.V[l] / model.t0[l])
        amps.append(model.r[l] * trans)
        trans *= 1.0 - model.r[l] ** 2
    for a in range(L):
        for c in range(L):
            for b in range(min(a, c)):
                t0 = model.t0[a] + model.t0[c] - model.t0[b]
                t0s.append(t0)
                v2s.append((model.V[a] + model.V[c] - model.V[b]) / t0)
                amps.append(-model.r[a] * model.r[b] * model.r[c])
    return np.array(t0s), np.array(v2s), np.array(amps)


def ricker(u: np.ndarray, fpeak: float, half_support: float) -> np.ndarray:
    a = (math.pi * fpeak) ** 2 * u * u
    w = (1.0 - 2.0 * a) * np.exp(-a)
    return np.where(np.abs(u) <= half_support, w, 0.0)


def base_traces(cfg: Config) -> np.ndarray:
    """[n][nt] fp32: the noise-free trace for every |s - r| (the medium is laterally invariant), A_R applied.

    The kernels never exploit this Toeplitz structure; it only makes the generator cheap."""
    model = layer_model(cfg)
    t0, v2, amp = _events(model)
    t = np.arange(cfg.nt) * cfg.dt
    tmax = (cfg.nt // 2) * cfg.dt
    out = np.zeros((cfg.n, cfg.nt), dtype=np.float64)
    for off_i in range(cfg.n):
        off = off_i * cfg.dx
        tau = np.sqrt(t0 * t0 + off * off / v2)
        keep = tau + cfg.half_support <= tmax
        a = amp * t0 / tau
        for tk, ak in zip(tau[keep], a[keep]):
            j0 = max(0, int(math.floor((tk - cfg.half_support) / cfg.dt)) - 1)
            j1 = min(cfg.nt // 2, int(math.ceil((tk + cfg.half_support) / cfg.dt)) + 2)
            out[off_i, j0:j1] += ak * ricker(t[j0:j1] - tk, cfg.fpeak, cfg.half_support)
    return (cfg.A_R * out).astype(np.float32)


def _noise_sigma(cfg: Config, base: np.ndarray) -> np.ndarray:
    half = cfg.nt // 2
    rms = np.sqrt(np.mean(base[:, :half].astype(np.float64) ** 2, axis=1))
    return rms * 10.0 ** (-cfg.noise_snr_db / 20.0)


def _noise_block(cfg: Config, shots: np.ndarray, recs: np.ndarray) -> np.ndarray:
    """Standard normals [ns][nr][nt/2] by Box-Muller; a pure function of (seed, s, r, sample)."""
    half = cfg.nt // 2
    pairs = half // 2
    trace_id = shots.astype(_U64)[:, None] * _U64(cfg.n) + recs.astype(_U64)[None, :]
    ctr = trace_id[:, :, None] * _U64(half) + (_U64(2) * np.arange(pairs, dtype=_U64))[None, None, :]
    u1 = 1.0 - uniforms(cfg.seed, _S_NOISE, ctr)                 # (0, 1]
    u2 = uniforms(cfg.seed, _S_NOISE, ctr + _U64(1))
    rad = np.sqrt(-2.0 * np.log(u1))
    ang = 2.0 * math.pi * u2
    z = np.empty(trace_id.shape + (half,), dtype=np.float64)
    z[..., 0::2] = rad * np.cos(ang)
    z[..., 1::2] = rad * np.sin(ang)
    return z


def R_block(cfg: Config, base: np.ndarray, shots, recs) -> np.ndarray:
    """[len(shots)][len(recs)][nt] fp32 time-domain reflection response R(x_R = r, x = s, t)."""
    shots = np.asarray(shots, dtype=np.int64)
    recs = np.asarray(recs, dtype=np.int64)
    off = np.abs(shots[:, None] - recs[None, :])
    blk = base[off]                                              # gather (copy)
    if cfg.noise_snr_db is not None:
        sigma = _noise_sigma(cfg, base)[off]
        half = cfg.nt // 2
        z = _noise_block(cfg, shots, recs)
        blk[:, :, :half] = (blk[:, :, :half].astype(np.float64) + sigma[:, :, None] * z).astype(np.float32)
    return blk


def R_full(cfg: Config, base: np.ndarray | None = None) -> np.ndarray:
    """The whole [n][n][nt] fp32 cube (configs 0-2 on the host; larger configs use R_block chunks)."""
    if base is None:
        base = base_traces(cfg)
    idx = np.arange(cfg.n)
    return R_block(cfg, base, idx, idx)


# ----------------------------------------------------------------------------------------------
# focal points, first arrivals
# ----------------------------------------------------------------------------------------------
def focal_points(cfg: Config):
    """(x_F[nfoc], z_F[nfoc]) in metres (laterals are relative to the spread)."""
    rule = cfg.focal.split(":")
    n, dx, nf = cfg.n, cfg.dx, cfg.nfoc
    if rule[0] == "single":                       # one point under the centre receiver
        assert nf == 1
        xf, zf = np.array([0.5 * (n - 1) * dx]), np.array([float(rule[1])])
    elif rule[0] == "line":                       # one focal point under every receiver
        assert nf == n
        xf, zf = np.arange(n) * dx, np.full(n, float(rule[1]))
    elif rule[0] == "grid8x8":                    # 8 depths x 8 laterals over the central half of the spread
        assert nf == 64
        depths = 400.0 + 200.0 * np.arange(8)
        lat = np.round((n - 1) * (0.25 + 0.0715 * np.arange(8))) * dx     # n = 2001: indices 500 + 143 q
        zf, xf = [a.ravel() for a in np.meshgrid(depths, lat, indexing="ij")]
    elif rule[0] == "line256":                    # 256 points, 10 dx apart, centred
        assert nf == 256
        xf = 0.5 * (n - 1) * dx + (np.arange(256) - 127.5) * 10.0 * dx
        zf = np.full(256, float(rule[1]))
    elif rule[0] == "fan":                        # reduced test copies: nfoc points over the central half, 8 depths
        f = np.arange(nf)
        xf = (0.25 + 0.5 * (f + 0.5) / nf) * (n - 1) * dx
        zf = float(rule[1]) + 100.0 * (f % 8)
    else:
        raise ValueError(cfg.focal)
    return xf.astype(np.float64), zf.astype(np.float64)


def first_arrivals(cfg: Config, focs=None, recs=None):
    """G_d[f][r][nt] fp32 and t_d[f][r] fp32 (seconds) for the chosen focal points / receivers."""
    xf, zf = focal_points(cfg)
    if focs is not None:
        focs = np.asarray(focs, dtype=np.int64)
        xf, zf = xf[focs], zf[focs]
    r = np.arange(cfg.n) if recs is None else np.asarray(recs, dtype=np.int64)
    v0 = layer_model(cfg).v[0]
    td = np.sqrt(zf[:, None] ** 2 + (r[None, :] * cfg.dx - xf[:, None]) ** 2) / v0
    # keep clear of exact half-sample ties of t_d/dt
    frac = td / cfg.dt + 0.5
    tie = np.abs(frac - np.round(frac)) < 1e-3
    td = np.where(tie, td + 0.01 * cfg.dt, td)
    td32 = td.astype(np.float32)
    t = np.arange(cfg.nt) * cfg.dt
    tmax = (cfg.nt // 2) * cfg.dt
    live = (td32.astype(np.float64) + cfg.half_support <= tmax)
    gd = np.zeros(td.shape + (cfg.nt,), dtype=np.float32)
    for f in range(td.shape[0]):
        u = t[None, :] - td32[f].astype(np.float64)[:, None]
        gd[f] = (ricker(u, cfg.fpeak, cfg.half_support) * live[f][:, None]).astype(np.float32)
    return gd, td32


def subset_indices(cfg: Config, nrec: int = 32, nfoc: int = 16):
    """Seeded sample without replacement of receiver / focal indices (seed_k + 1000)."""
    rng = np.random.Generator(np.random.PCG64(cfg.seed + 1000))
    recs = np.sort(rng.choice(cfg.n, size=min(nrec, cfg.n), replace=False))
    focs = np.sort(rng.choice(cfg.nfoc, size=min(nfoc, cfg.nfoc), replace=False))
    return recs, focs


# ----------------------------------------------------------------------------------------------
# device twin of R_block: configs 3 and 4 (33 GB / 250 GB of time-domain R) are produced chunk by chunk on the device
# and handed to mk_load_R; nothing of that size is ever stored.  Same recipe, same counters: a gather of the same base
# traces plus (config 3) the same Box-Muller normals.  Still no arithmetic of the method.
# ----------------------------------------------------------------------------------------------
def _i64(v: int) -> int:
    """a uint64 constant as the int64 with the same bits (torch has no uint64 arithmetic)."""
    v &= (1 << 64) - 1
    return v - (1 << 64) if v >= (1 << 63) else v


def _mix_torch(x):
    """_mix on int64 tensors: wrapping multiply, logical right shifts by masking the sign extension."""
    def lsr(z, k):
        return (z >> k) & ((1 << (64 - k)) - 1)
    z = x + _i64(int(_GOLD))
    z = (z ^ lsr(z, 30)) * _i64(int(_M1))
    z = (z ^ lsr(z, 27)) * _i64(int(_M2))
    return z ^ lsr(z, 31)


def _uniforms_torch(seed: int, stream: int, idx):
    import torch
    z = _mix_torch(idx * _i64(int(_GOLD)) + _i64(int(_key(seed, stream))))
    top53 = (z >> 11) & ((1 << 53) - 1)
    return top53.to(torch.float64) * (1.0 / 9007199254740992.0)


class DeviceR:
    """R_block on a torch device.  `take(shots)` returns the fp32 chunk [len(shots)][n][nt] (receivers = all)."""

    def __init__(self, cfg: Config, device, base: np.ndarray | None = None):
        import torch
        self.cfg, self.device = cfg, device
        base = base_traces(cfg) if base is None else base
        self.base = torch.from_numpy(base).to(device)
        self.sigma = None
        if cfg.noise_snr_db is not None:
            self.sigma = torch.from_numpy(_noise_sigma(cfg, base)).to(device)          # fp64 [n]

    def take(self, shots, recs=None):
        import torch
        cfg = self.cfg
        shots = torch.as_tensor(np.asarray(shots, dtype=np.int64), device=self.device)
        recs = torch.arange(cfg.n, device=self.device) if recs is None else torch.as_tensor(np.asarray(recs, dtype=np.int64),
                                                                                          device=self.device)
        off = (shots[:, None] - recs[None, :]).abs()
        blk = self.base[off]                                                           # gather (copy)
        if self.sigma is not None:
            half, pairs = cfg.nt // 2, cfg.nt // 4
            trace_id = shots[:, None] * cfg.n + recs[None, :]
            ctr = trace_id[:, :, None] * half + 2 * torch.arange(pairs, device=self.device, dtype=torch.int64)[None, None, :]
            u1 = 1.0 - _uniforms_torch(cfg.seed, _S_NOISE, ctr)
            u2 = _uniforms_torch(cfg.seed, _S_NOISE, ctr + 1)
            rad = torch.sqrt(-2.0 * torch.log(u1))
            ang = 2.0 * math.pi * u2
            z = torch.empty(trace_id.shape + (half,), dtype=torch.float64, device=self.device)
            z[..., 0::2] = rad * torch.cos(ang)
            z[..., 1::2] = rad * torch.sin(ang)
            blk[:, :, :half] = (blk[:, :, :half].to(torch.float64) + self.sigma[off][:, :, None] * z).to(torch.float32)
        return blk


def first_arrivals_torch(cfg: Config, device, focs=None, chunk: int = 8):
    """first_arrivals with the wavelet evaluated on `device` (config 4: 256 x 3901 x 4096 samples).  t_d is the
    host function's, bit for bit; G_d may differ from the numpy one in the last fp32 bit (exp), so whoever needs
    the same bytes on both sides takes them from this tensor."""
    import torch
    xf, zf = focal_points(cfg)
    if focs is not None:
        focs = np.asarray(focs, dtype=np.int64)
        xf, zf = xf[focs], zf[focs]
    r = np.arange(cfg.n)
    v0 = layer_model(cfg).v[0]
    td = np.sqrt(zf[:, None] ** 2 + (r[None, :] * cfg.dx - xf[:, None]) ** 2) / v0
    frac = td / cfg.dt + 0.5
    tie = np.abs(frac - np.round(frac)) < 1e-3
    td32 = np.where(tie, td + 0.01 * cfg.dt, td).astype(np.float32)
    tmax = (cfg.nt // 2) * cfg.dt
    d_td = torch.from_numpy(td32).to(device)
    t = torch.arange(cfg.nt, device=device, dtype=torch.float64) * cfg.dt
    gd = torch.empty((len(xf), cfg.n, cfg.nt), dtype=torch.float32, device=device)
    for f0 in range(0, len(xf), chunk):
        tdc = d_td[f0:f0 + chunk].to(torch.float64)
        u = t[None, None, :] - tdc[:, :, None]
        a = (math.pi * cfg.fpeak) ** 2 * u * u
        w = (1.0 - 2.0 * a) * torch.exp(-a)
        w = torch.where(u.abs() <= cfg.half_support, w, torch.zeros_like(w))
        live = (tdc + cfg.half_support <= tmax)
        gd[f0:f0 + chunk] = (w * live[:, :, None]).to(torch.float32)
    return gd, d_td

// mk_fft_kernels.cu — the per-trace kernels of the path:
//   k_window   h = clamp(floor(t_d/dt + 0.5) - eps, 0, nt/2)                                   (a4 table; G2c)
//   k_load_R   rFFT over t, keep B, fold dt*w[s], transpose to R^[r][k][s]                     (a0)
//   k_fwd      time field -> N^ band (optionally of the time-reversed field, optionally storing T src)   (a1, a6)
//   k_inv      spectrum -> time field with a linear epilogue (finals, bare synthesis)          (a3, a7)
//   k_post     p^ += S^; inverse rFFT; N_i = -Theta T S; f1min / f1plus accumulation; rFFT -> N^_i   (a3..a6 fused:
//              one pass over N per iteration, BASELINE.json north_star (c))
//
// Work decomposition.  One CTA (256 threads) owns one receiver r and FT consecutive focal points (FT a power of two
// <= 8), so the S^[r][k][f..] reads and the N^[k][r][f..] writes are contiguous 8*FT-byte segments.  The traces live
// in padded shared memory (fft_core.cuh).  Inside the CTA every trace belongs to a GROUP of 256/FT threads (one warp
// when FT = 8): the FFT passes, the window and the accumulation of a trace synchronise only inside its group
// (__syncwarp / a named barrier), so the groups drift apart and hide each other's latency; the CTA synchronises only
// around the two phases whose thread mapping crosses traces (spectrum load, spectrum store).
#include "mk_fft_common.cuh"

namespace mk {

using mkfft::Plan;

namespace {

constexpr int kThreads = 256;

struct Group {
  int tl;     // trace (local focal index) this thread works on
  int lane;   // index inside the group
  int size;   // threads per group = kThreads / FT
};

__device__ __forceinline__ Group my_group(int lgFT) {
  Group g;
  g.size = kThreads >> lgFT;
  g.tl = threadIdx.x / g.size;
  g.lane = threadIdx.x - g.tl * g.size;
  return g;
}

__device__ __forceinline__ void group_sync(const Group& g) {
  if (g.size == 32) __syncwarp();
  else if (g.size == kThreads) __syncthreads();
  else {  // FT = 2 or 4: named barriers 1..4 (immediate ids, so that only these are reserved)
    switch (g.tl) {
      case 0: asm volatile("bar.sync 1, %0;" ::"r"(g.size) : "memory"); break;
      case 1: asm volatile("bar.sync 2, %0;" ::"r"(g.size) : "memory"); break;
      case 2: asm volatile("bar.sync 3, %0;" ::"r"(g.size) : "memory"); break;
      default: asm volatile("bar.sync 4, %0;" ::"r"(g.size) : "memory"); break;
    }
  }
}

// forward passes of ONE trace by its group (decimation in frequency; leaves Z digit-reversed)
__device__ __forceinline__ void fft_fwd(float2* z, const Plan& p, const float2* __restrict__ tw, const Group& g) {
  for (int ps = 0; ps < p.npass; ++ps) {
    const int lgr = p.lgr[ps], lgL = p.lgL[ps], nb = p.M >> lgr;
    if (lgr == 3) {
      for (int b = g.lane; b < nb; b += g.size) mkfft::fwd_butterfly<3>(z, tw, p.nt, lgL, b);
    } else if (lgr == 2) {
      for (int b = g.lane; b < nb; b += g.size) mkfft::fwd_butterfly<2>(z, tw, p.nt, lgL, b);
    } else {
      for (int b = g.lane; b < nb; b += g.size) mkfft::fwd_butterfly<1>(z, tw, p.nt, lgL, b);
    }
    group_sync(g);
  }
}

__device__ __forceinline__ void fft_inv(float2* z, const Plan& p, const float2* __restrict__ tw, const Group& g) {
  for (int ps = p.npass - 1; ps >= 0; --ps) {
    const int lgr = p.lgr[ps], lgL = p.lgL[ps], nb = p.M >> lgr;
    if (lgr == 3) {
      for (int b = g.lane; b < nb; b += g.size) mkfft::inv_butterfly<3>(z, tw, p.nt, lgL, b);
    } else if (lgr == 2) {
      for (int b = g.lane; b < nb; b += g.size) mkfft::inv_butterfly<2>(z, tw, p.nt, lgL, b);
    } else {
      for (int b = g.lane; b < nb; b += g.size) mkfft::inv_butterfly<1>(z, tw, p.nt, lgL, b);
    }
    group_sync(g);
  }
}

// the group's trace: contiguous-time fp32 source -> padded buffer (float4 loads, 4 in flight per thread)
__device__ __forceinline__ void load_trace(float2* z, const float* __restrict__ src, int nt, const Group& g) {
  const float4* s4 = reinterpret_cast<const float4*>(src);
  const int q = nt >> 2;
  for (int j0 = g.lane; j0 < q; j0 += 4 * g.size) {
    float4 v[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int j4 = j0 + u * g.size;
      if (j4 < q) v[u] = __ldg(s4 + j4);
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int j4 = j0 + u * g.size;
      if (j4 < q) {
        z[mkfft::padi(2 * j4)] = make_float2(v[u].x, v[u].y);
        z[mkfft::padi(2 * j4 + 1)] = make_float2(v[u].z, v[u].w);
      }
    }
  }
}

__device__ __forceinline__ float4 read4(const float2* z, int j4) {  // samples 4 j4 .. 4 j4 + 3 of the padded trace
  const float2 a = z[mkfft::padi(2 * j4)], b = z[mkfft::padi(2 * j4 + 1)];
  return make_float4(a.x, a.y, b.x, b.y);
}
__device__ __forceinline__ void write4(float2* z, int j4, float4 v) {
  z[mkfft::padi(2 * j4)] = make_float2(v.x, v.y);
  z[mkfft::padi(2 * j4 + 1)] = make_float2(v.z, v.w);
}
// time-reversed samples: (T u)[4 j4 + e] = u[(nt - 4 j4 - e) % nt], e = 0..3
__device__ __forceinline__ float4 read4_reversed(const float2* z, int j4, int nt) {
  const float* zf = reinterpret_cast<const float*>(z);
  const int j = 4 * j4;
  return make_float4(zf[mkfft::padj((nt - j) & (nt - 1))], zf[mkfft::padj(nt - j - 1)], zf[mkfft::padj(nt - j - 2)],
                     zf[mkfft::padj(nt - j - 3)]);
}

// Z (digit-reversed, scaled) of all FT traces from their band-limited half spectra.  CTA-wide: consecutive threads
// take consecutive focal points of one bin.  load(tl, kk, aux) returns X[klo + kk] of trace tl (and may fetch a side
// value into aux); commit(tl, kk, X, aux) runs afterwards.  Both are called exactly once per in-band (k, tl); the
// loads of four items are issued before anything is consumed.
template <bool CONJ, typename Load, typename Commit>
__device__ __forceinline__ void spectrum_to_Z(float2* smem, int nf, int lgFT, int MP, const Plan& p,
                                              const float2* __restrict__ tw, int klo, int nb, Load load, Commit commit) {
  const int M = p.M, half = M >> 1, FT = 1 << lgFT;
  const float scale = 1.0f / (2.0f * (float)M);
  const int total = (half + 1) << lgFT;
  for (int i0 = threadIdx.x; i0 < total; i0 += 4 * kThreads) {
    float2 a[4], b[4], xa[4], xb[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int idx = i0 + u * kThreads;
      a[u] = b[u] = xa[u] = xb[u] = make_float2(0.f, 0.f);
      if (idx < total) {
        const int k = idx >> lgFT, tl = idx & (FT - 1), k2 = M - k;
        if (tl < nf) {
          if (k >= klo && k < klo + nb) a[u] = load(tl, k - klo, xa[u]);
          if (k2 != k && k2 >= klo && k2 < klo + nb) b[u] = load(tl, k2 - klo, xb[u]);
        }
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int idx = i0 + u * kThreads;
      if (idx >= total) continue;
      const int k = idx >> lgFT, tl = idx & (FT - 1), k2 = M - k;
      if (tl >= nf) continue;
      if (k >= klo && k < klo + nb) commit(tl, k - klo, a[u], xa[u]);
      if (k2 != k && k2 >= klo && k2 < klo + nb) commit(tl, k2 - klo, b[u], xb[u]);
      float2 x = a[u], y = b[u];
      if (k2 == k) y = x;
      if (k == 0) {  // DC and Nyquist are real for a real trace (irfft convention)
        x.y = 0.f;
        y.y = 0.f;
      }
      if (CONJ) {
        x.y = -x.y;
        y.y = -y.y;
      }
      float2* zt = smem + tl * MP;
      zt[mkfft::padi(mkfft::freq_pos(p, k))] = mkfft::irfft_pre(x, y, tw[k], scale);
      if (k2 < M && k2 != k) zt[mkfft::padi(mkfft::freq_pos(p, k2))] = mkfft::irfft_pre(y, x, tw[k2], scale);
    }
  }
}

// band of the half spectra of all FT traces (held digit-reversed in smem) -> operand; CTA-wide mapping
__device__ __forceinline__ void Z_to_operand(const float2* smem, int nf, int lgFT, int MP, const FftParams& P, int r, int f0,
                                             bool conj_out, const OperandOut& O) {
  const int FT = 1 << lgFT, total = P.nb << lgFT;
  for (int idx = threadIdx.x; idx < total; idx += kThreads) {
    const int kk = idx >> lgFT, tl = idx & (FT - 1);
    if (tl >= nf) continue;
    float2 X = mkfft::rfft_bin(smem + tl * MP, P.plan, P.tw, P.klo + kk);
    if (conj_out) X.y = -X.y;  // spectrum of the time-reversed real trace
    store_operand(O, P.ld, kk, r, f0 + tl, X);
  }
}

// ------------------------------------------------------------------------------------------------ k_window
__global__ void k_window(const float* __restrict__ td, int* __restrict__ h, int ntr, double dt, int eps, int nt) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= ntr) return;
  const double m = floor((double)td[i] / dt + 0.5);
  double hv = m - (double)eps;
  hv = fmax(hv, 0.0);
  hv = fmin(hv, (double)(nt / 2));
  h[i] = (int)hv;
}

// ------------------------------------------------------------------------------------------------ k_load_R
// grid (ceil(nshots/ST), nrec); Rt: [nshots][nrec][nt]
__global__ void __launch_bounds__(kThreads) k_load_R(const float* __restrict__ Rt, float2* __restrict__ Rhat, FftParams P,
                                                     int shot0, int nshots, int lgST) {
  extern __shared__ float2 smem[];
  const int MP = mkfft::padded_len(P.plan.M), ST = 1 << lgST;
  const int r = P.r0 + blockIdx.y, g0 = blockIdx.x * ST;
  const int ns = min(ST, nshots - g0);
  const Group g = my_group(lgST);
  const size_t nt = P.plan.nt;
  if (g.tl < ns) {
    float2* z = smem + g.tl * MP;
    load_trace(z, Rt + ((size_t)(g0 + g.tl) * P.n + r) * nt, P.plan.nt, g);
    group_sync(g);
    fft_fwd(z, P.plan, P.tw, g);
  }
  __syncthreads();
  const int total = P.nb << lgST;
  for (int idx = threadIdx.x; idx < total; idx += kThreads) {
    const int kk = idx >> lgST, tl = idx & (ST - 1);
    if (tl >= ns) continue;
    const int s = shot0 + g0 + tl;
    const float sc = __ldg(P.wscale + s);
    const float2 X = mkfft::rfft_bin(smem + tl * MP, P.plan, P.tw, P.klo + kk);
    Rhat[rhat_index(P.tiled, r - P.r0, kk, s, P.nb, P.ld)] = make_float2(sc * X.x, sc * X.y);
  }
}

// ------------------------------------------------------------------------------------------------ k_fwd
// grid (ceil(nfoc/FT), n); src: [nfoc][n][nt]
__global__ void __launch_bounds__(kThreads) k_fwd(const float* __restrict__ src, const __grid_constant__ OperandOut O, FftParams P, int lgFT,
                                                  int conj_out, float* __restrict__ init_Tsrc) {
  extern __shared__ float2 smem[];
  const int MP = mkfft::padded_len(P.plan.M), FT = 1 << lgFT;
  const int r = P.r0 + blockIdx.y, f0 = blockIdx.x * FT;
  const int nf = min(FT, P.nfoc - f0);
  const int nt = P.plan.nt;
  const Group g = my_group(lgFT);
  if (g.tl < nf) {
    float2* z = smem + g.tl * MP;
    const size_t base = ((size_t)(f0 + g.tl) * P.n + r) * nt;
    load_trace(z, src + base, nt, g);
    group_sync(g);
    if (init_Tsrc) {  // f1plus = N_{-1} = T G_d   [PAPER.md:19, 67, 74]
      float4* dst = reinterpret_cast<float4*>(init_Tsrc + base);
      for (int j4 = g.lane; j4 < (nt >> 2); j4 += g.size) dst[j4] = read4_reversed(z, j4, nt);
      group_sync(g);  // the in-place FFT below overwrites what this loop reads
    }
    fft_fwd(z, P.plan, P.tw, g);
  }
  __syncthreads();
  Z_to_operand(smem, nf, lgFT, MP, P, r, f0, conj_out != 0, O);
}

// ------------------------------------------------------------------------------------------------ k_inv
// grid (ceil(nfoc/FT), n); spec: [n][nb][ldf]; out[j] = sS*S[j] + sA*A[j] + sB*B[(nt-j)%nt]
__global__ void __launch_bounds__(kThreads) k_inv(const float2* __restrict__ spec, FftParams P, int lgFT, float* __restrict__ out,
                                                  float sS, const float* __restrict__ A, float sA,
                                                  const float* __restrict__ B, float sB) {
  extern __shared__ float2 smem[];
  const int MP = mkfft::padded_len(P.plan.M), FT = 1 << lgFT;
  const int r = P.r0 + blockIdx.y, f0 = blockIdx.x * FT;
  const int nf = min(FT, P.nfoc - f0);
  const int nt = P.plan.nt;
  const float2* srow = spec + (size_t)r * P.nb * P.ldf + f0;
  spectrum_to_Z<false>(smem, nf, lgFT, MP, P.plan, P.tw, P.klo, P.nb,
                       [&](int tl, int kk, float2&) { return __ldg(srow + (size_t)kk * P.ldf + tl); },
                       [](int, int, float2, float2) {});
  __syncthreads();
  const Group g = my_group(lgFT);
  if (g.tl >= nf) return;
  float2* z = smem + g.tl * MP;
  fft_inv(z, P.plan, P.tw, g);
  const size_t base = ((size_t)(f0 + g.tl) * P.n + r) * nt;
  const float4* A4 = A ? reinterpret_cast<const float4*>(A + base) : nullptr;
  float4* o4 = reinterpret_cast<float4*>(out + base);
  for (int j4 = g.lane; j4 < (nt >> 2); j4 += g.size) {
    float4 v = read4(z, j4);
    v = make_float4(sS * v.x, sS * v.y, sS * v.z, sS * v.w);
    if (A4) {
      const float4 a = __ldg(A4 + j4);
      v.x += sA * a.x;
      v.y += sA * a.y;
      v.z += sA * a.z;
      v.w += sA * a.w;
    }
    if (B) {
      const int j = 4 * j4;
      v.x += sB * __ldg(B + base + ((nt - j) & (nt - 1)));
      v.y += sB * __ldg(B + base + (nt - j - 1));
      v.z += sB * __ldg(B + base + (nt - j - 2));
      v.w += sB * __ldg(B + base + (nt - j - 3));
    }
    o4[j4] = v;
  }
}

// ------------------------------------------------------------------------------------------------ k_post
// grid (ceil(nfoc/FT), n).  Shat, phat: [n][nb][ldf]; operand out: see store_operand; h: [nfoc][n];
// f1plus / f1min: [nfoc][n][nt]
__global__ void __launch_bounds__(kThreads) k_post(const float2* __restrict__ Shat, float2* __restrict__ phat, const __grid_constant__ OperandOut O,
                                                   const int* __restrict__ h, float* __restrict__ f1plus, float* __restrict__ f1min,
                                                   FftParams P, int lgFT, int parity_even, float* __restrict__ Ni_out) {
  extern __shared__ float2 smem[];
  const int MP = mkfft::padded_len(P.plan.M), FT = 1 << lgFT;
  const int r = P.r0 + blockIdx.y, f0 = blockIdx.x * FT;
  const int nf = min(FT, P.nfoc - f0);
  const int nt = P.plan.nt;
  const size_t rowoff = (size_t)r * P.nb * P.ldf + f0;
  // a3: p^ += S^ ; Z of conj(S^) so that the inverse transform yields u = T S directly  [PAPER.md:79, 71]
  spectrum_to_Z<true>(
      smem, nf, lgFT, MP, P.plan, P.tw, P.klo, P.nb,
      [&](int tl, int kk, float2& pv) {
        const size_t o = rowoff + (size_t)kk * P.ldf + tl;
        pv = phat[o];
        return __ldg(Shat + o);
      },
      [&](int tl, int kk, float2 s, float2 pv) { phat[rowoff + (size_t)kk * P.ldf + tl] = make_float2(pv.x + s.x, pv.y + s.y); });
  __syncthreads();
  const Group g = my_group(lgFT);
  if (g.tl < nf) {
    float2* z = smem + g.tl * MP;
    fft_inv(z, P.plan, P.tw, g);  // z = u = T S
    const int hh = __ldg(h + (size_t)(f0 + g.tl) * P.n + r);
    const size_t base = ((size_t)(f0 + g.tl) * P.n + r) * nt;
    const int q = nt >> 2;
    // a5: N_i = -Theta u.  i even: f1min -= T N_i  <=>  f1min[j] += Theta[j] u[(nt-j)%nt];  i odd: f1plus += N_i
    //     [PAPER.md:82-85].  Theta[j] = 1 iff j < h or j > nt - h; only chunks that meet the window touch HBM.
    float4* acc4 = reinterpret_cast<float4*>((parity_even ? f1min : f1plus) + base);
    for (int j4 = g.lane; j4 < q; j4 += g.size) {
      const int j = 4 * j4;
      if (!(j < hh || j + 3 > nt - hh)) continue;
      const float4 u = parity_even ? read4_reversed(z, j4, nt) : read4(z, j4);
      float4 a = acc4[j4];
      const float sg = parity_even ? 1.f : -1.f;
      if (j < hh || j > nt - hh) a.x += sg * u.x;
      if (j + 1 < hh || j + 1 > nt - hh) a.y += sg * u.y;
      if (j + 2 < hh || j + 2 > nt - hh) a.z += sg * u.z;
      if (j + 3 < hh || j + 3 > nt - hh) a.w += sg * u.w;
      acc4[j4] = a;
    }
    group_sync(g);
    // a4: N_i in place (hard 0/1 window, strict inequality; G2)
    float4* ni4 = Ni_out ? reinterpret_cast<float4*>(Ni_out + base) : nullptr;
    for (int j4 = g.lane; j4 < q; j4 += g.size) {
      const int j = 4 * j4;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (j < hh || j + 3 > nt - hh) {
        const float4 u = read4(z, j4);
        v.x = (j < hh || j > nt - hh) ? -u.x : 0.f;
        v.y = (j + 1 < hh || j + 1 > nt - hh) ? -u.y : 0.f;
        v.z = (j + 2 < hh || j + 2 > nt - hh) ? -u.z : 0.f;
        v.w = (j + 3 < hh || j + 3 > nt - hh) ? -u.w : 0.f;
      }
      write4(z, j4, v);
      if (ni4) ni4[j4] = v;
    }
    group_sync(g);
    fft_fwd(z, P.plan, P.tw, g);  // a6
  }
  __syncthreads();
  Z_to_operand(smem, nf, lgFT, MP, P, r, f0, false, O);
}

int pick_lgft(const mk_ctx* c, int count) {
  const size_t per = (size_t)mkfft::padded_len(c->plan.M) * sizeof(float2);
  int lg = 3;                                           // FT <= 8
  while (lg > 0 && ((size_t)1 << lg) * per > 72000) --lg;  // <= ~70 KB of traces per CTA: 3 CTAs per SM
  while (lg > 0 && (1 << (lg - 1)) >= count) --lg;      // no more slots than traces
  return lg;
}

FftParams make_params(const mk_ctx* c, int nfoc, int ldf) {
  FftParams P;
  P.plan = c->plan;
  P.tw = c->d_tw;
  P.n = c->n;
  P.wscale = c->d_wscale;
  P.nb = c->nb;
  P.klo = c->klo;
  P.ld = c->ld;
  P.ldf = ldf;
  P.nfoc = nfoc;
  P.tiled = c->rhat_layout;
  P.r0 = c->r0;
  return P;
}

template <typename K>
int set_smem(mk_ctx* c, K kernel, size_t bytes) {
  if (bytes > c->smem_optin) return set_err(c, MK_ERR_INVALID_ARG, "trace too long for shared memory");
  return check_cuda(c, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes), "cudaFuncSetAttribute");
}

size_t trace_smem(const mk_ctx* c, int lgft) { return ((size_t)mkfft::padded_len(c->plan.M) << lgft) * sizeof(float2); }

}  // namespace

int launch_window(mk_ctx* c, const float* d_td, int* d_h, int ntr) {
  k_window<<<(ntr + 255) / 256, 256, 0, c->stream>>>(d_td, d_h, ntr, c->dt, c->eps, c->nt);
  ++c->launches;
  return check_cuda(c, cudaGetLastError(), "k_window");
}

int launch_load_R(mk_ctx* c, const RowBlock& rb, const float* d_R_time, int shot0, int nshots) {
  if (fast_fft_ok(c)) return launch_load_R_fast(c, rb, d_R_time, shot0, nshots);
  const int lg = pick_lgft(c, nshots), ST = 1 << lg;
  const size_t smem = trace_smem(c, lg);
  if (int rc = set_smem(c, k_load_R, smem)) return rc;
  const dim3 grid((nshots + ST - 1) / ST, rb.nrow);
  FftParams P = make_params(c, 0, 0);
  P.r0 = rb.r0;
  if (rb.ld) P.ld = rb.ld;
  if (rb.src_n) P.n = rb.src_n;
  k_load_R<<<grid, kThreads, smem, c->stream>>>(d_R_time, rb.Rhat, P, shot0, nshots, lg);
  ++c->launches;
  return check_cuda(c, cudaGetLastError(), "k_load_R");
}

int launch_fwd(mk_ctx* c, const float* d_src, const OperandOut& O, int nfoc, bool conj_out, float* d_init_Tsrc) {
  if (fast_fft_ok(c)) return launch_fwd_fast(c, d_src, O, nfoc, conj_out, d_init_Tsrc);
  const int lg = pick_lgft(c, nfoc), FT = 1 << lg;
  const size_t smem = trace_smem(c, lg);
  if (int rc = set_smem(c, k_fwd, smem)) return rc;
  const dim3 grid((nfoc + FT - 1) / FT, c->nrow);
  k_fwd<<<grid, kThreads, smem, c->stream>>>(d_src, O, make_params(c, nfoc, O.ldf), lg, conj_out ? 1 : 0, d_init_Tsrc);
  ++c->launches;
  return check_cuda(c, cudaGetLastError(), "k_fwd");
}

int launch_inv(mk_ctx* c, const float2* d_spec, int nfoc, int ldf, float* d_out, float sS, const float* d_A, float sA,
               const float* d_B, float sB) {
  if (fast_fft_ok(c)) return launch_inv_fast(c, d_spec, nfoc, ldf, d_out, sS, d_A, sA, d_B, sB);
  const int lg = pick_lgft(c, nfoc), FT = 1 << lg;
  const size_t smem = trace_smem(c, lg);
  if (int rc = set_smem(c, k_inv, smem)) return rc;
  const dim3 grid((nfoc + FT - 1) / FT, c->nrow);
  k_inv<<<grid, kThreads, smem, c->stream>>>(d_spec, make_params(c, nfoc, ldf), lg, d_out, sS, d_A, sA, d_B, sB);
  ++c->launches;
  return check_cuda(c, cudaGetLastError(), "k_inv");
}

int launch_post(mk_ctx* c, const OperandOut& O, int parity_even, float* d_Ni_out) {
  if (fast_fft_ok(c)) return launch_post_fast(c, O, parity_even, d_Ni_out);
  const int lg = pick_lgft(c, c->nfoc), FT = 1 << lg;
  const size_t smem = trace_smem(c, lg);
  if (int rc = set_smem(c, k_post, smem)) return rc;
  const dim3 grid((c->nfoc + FT - 1) / FT, c->nrow);
  k_post<<<grid, kThreads, smem, c->stream>>>(c->d_Shat, c->d_phat, O, c->d_h, c->acc_plus, c->acc_min,
                                              make_params(c, c->nfoc, c->ldf), lg, parity_even, d_Ni_out);
  ++c->launches;
  return check_cuda(c, cudaGetLastError(), "k_post");
}

}  // namespace mk

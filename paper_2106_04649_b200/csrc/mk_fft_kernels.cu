// mk_fft_kernels.cu — the per-trace kernels of the path:
//   k_window   h = clamp(floor(t_d/dt + 0.5) - eps, 0, nt/2)                                   (a4 table; G2c)
//   k_load_R   rFFT over t, keep B, fold dt*w[s], transpose to R^[r][k][s]                     (a0)
//   k_fwd      time field -> N^ band (optionally of the time-reversed field, optionally storing T src)   (a1, a6)
//   k_inv      spectrum -> time field with a linear epilogue (finals, bare synthesis)          (a3, a7)
//   k_post     p^ += S^; inverse rFFT; N_i = -Theta T S; f1min / f1plus accumulation; rFFT -> N^_i   (a3..a6 fused:
//              one pass over N per iteration, BASELINE.json north_star (c))
// One CTA owns one receiver r and FT consecutive focal points, so both the S^[r][k][f..] reads and the
// N^[k][r][f..] writes are contiguous 8*FT-byte segments.  Traces live in padded shared memory (fft_core.cuh).
#include "mk_internal.cuh"

namespace mk {

using mkfft::Plan;

namespace {

constexpr int kThreads = 256;

__device__ __forceinline__ void fft_batch_fwd(float2* z, int ntr, int MP, const Plan& p, const float2* __restrict__ tw) {
  for (int ps = 0; ps < p.npass; ++ps) {
    const int lgr = p.lgr[ps], lgL = p.lgL[ps], lgB = p.logM - lgr;
    const int total = ntr << lgB, mask = (1 << lgB) - 1;
    if (lgr == 3) {
      for (int b = threadIdx.x; b < total; b += blockDim.x) mkfft::fwd_butterfly<3>(z + (b >> lgB) * MP, tw, p.nt, lgL, b & mask);
    } else if (lgr == 2) {
      for (int b = threadIdx.x; b < total; b += blockDim.x) mkfft::fwd_butterfly<2>(z + (b >> lgB) * MP, tw, p.nt, lgL, b & mask);
    } else {
      for (int b = threadIdx.x; b < total; b += blockDim.x) mkfft::fwd_butterfly<1>(z + (b >> lgB) * MP, tw, p.nt, lgL, b & mask);
    }
    __syncthreads();
  }
}

__device__ __forceinline__ void fft_batch_inv(float2* z, int ntr, int MP, const Plan& p, const float2* __restrict__ tw) {
  for (int ps = p.npass - 1; ps >= 0; --ps) {
    const int lgr = p.lgr[ps], lgL = p.lgL[ps], lgB = p.logM - lgr;
    const int total = ntr << lgB, mask = (1 << lgB) - 1;
    if (lgr == 3) {
      for (int b = threadIdx.x; b < total; b += blockDim.x) mkfft::inv_butterfly<3>(z + (b >> lgB) * MP, tw, p.nt, lgL, b & mask);
    } else if (lgr == 2) {
      for (int b = threadIdx.x; b < total; b += blockDim.x) mkfft::inv_butterfly<2>(z + (b >> lgB) * MP, tw, p.nt, lgL, b & mask);
    } else {
      for (int b = threadIdx.x; b < total; b += blockDim.x) mkfft::inv_butterfly<1>(z + (b >> lgB) * MP, tw, p.nt, lgL, b & mask);
    }
    __syncthreads();
  }
}

// copy `ntr` contiguous-time traces into the padded buffers; src_of(tl) = pointer to trace tl
template <typename SrcOf>
__device__ __forceinline__ void load_traces(float2* z, int ntr, int MP, int nt, SrcOf src_of) {
  const int q = nt >> 2;  // float4 per trace
  for (int idx = threadIdx.x; idx < ntr * q; idx += blockDim.x) {
    const int tl = idx / q, j4 = idx - tl * q;
    const float4 v = __ldg(reinterpret_cast<const float4*>(src_of(tl)) + j4);
    float2* zt = z + tl * MP;
    zt[mkfft::padi(2 * j4)] = make_float2(v.x, v.y);
    zt[mkfft::padi(2 * j4 + 1)] = make_float2(v.z, v.w);
  }
}

// Build Z (digit-reversed, scaled) of `ntr` traces from a band-limited half spectrum.  spec_of(tl, kk) returns
// X[klo + kk] of trace tl (with every side effect the caller wants, e.g. the p^ accumulation).
template <bool CONJ, typename SpecOf>
__device__ __forceinline__ void spectrum_to_Z(float2* z, int ntr, int ft, int MP, const Plan& p, const float2* __restrict__ tw,
                                              int klo, int nb, SpecOf spec_of) {
  const int M = p.M, half = M >> 1;
  const float scale = 1.0f / (2.0f * (float)M);
  for (int idx = threadIdx.x; idx < (half + 1) * ft; idx += blockDim.x) {
    const int k = idx / ft, tl = idx - k * ft;
    if (tl >= ntr) continue;
    const int k2 = M - k;
    float2 a = make_float2(0.f, 0.f), b = make_float2(0.f, 0.f);
    if (k >= klo && k < klo + nb) a = spec_of(tl, k - klo);
    if (k2 != k && k2 >= klo && k2 < klo + nb) b = spec_of(tl, k2 - klo);
    if (k2 == k) b = a;
    if (k == 0) {  // DC and Nyquist are real for a real trace (irfft convention)
      a.y = 0.f;
      b.y = 0.f;
    }
    if (CONJ) {
      a.y = -a.y;
      b.y = -b.y;
    }
    float2* zt = z + tl * MP;
    zt[mkfft::padi(mkfft::freq_pos(p, k))] = mkfft::irfft_pre(a, b, tw[k], scale);
    if (k2 < M && k2 != k) zt[mkfft::padi(mkfft::freq_pos(p, k2))] = mkfft::irfft_pre(b, a, tw[k2], scale);
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
                                                     int shot0, int nshots, int ST, float scale_mid, float scale_end) {
  extern __shared__ float2 smem[];
  const int MP = mkfft::padded_len(P.plan.M);
  const int r = blockIdx.y, g0 = blockIdx.x * ST;
  const int ns = min(ST, nshots - g0);
  const size_t nt = P.plan.nt;
  load_traces(smem, ns, MP, P.plan.nt, [&](int tl) { return Rt + ((size_t)(g0 + tl) * P.n + r) * nt; });
  __syncthreads();
  fft_batch_fwd(smem, ns, MP, P.plan, P.tw);
  for (int idx = threadIdx.x; idx < P.nb * ST; idx += blockDim.x) {
    const int kk = idx / ST, tl = idx - kk * ST;
    if (tl >= ns) continue;
    const int s = shot0 + g0 + tl;
    const float sc = (P.n > 1 && (s == 0 || s == P.n - 1)) ? scale_end : scale_mid;
    const float2 X = mkfft::rfft_bin(smem + tl * MP, P.plan, P.tw, P.klo + kk);
    Rhat[((size_t)r * P.nb + kk) * P.ld + s] = make_float2(sc * X.x, sc * X.y);
  }
}

// ------------------------------------------------------------------------------------------------ k_fwd
// grid (ceil(nfoc/FT), n); src: [nfoc][n][nt]
__global__ void __launch_bounds__(kThreads) k_fwd(const float* __restrict__ src, float2* __restrict__ Nhat, FftParams P, int FT,
                                                  int conj_out, float* __restrict__ init_Tsrc) {
  extern __shared__ float2 smem[];
  const int MP = mkfft::padded_len(P.plan.M);
  const int r = blockIdx.y, f0 = blockIdx.x * FT;
  const int nf = min(FT, P.nfoc - f0);
  const int nt = P.plan.nt;
  load_traces(smem, nf, MP, nt, [&](int tl) { return src + ((size_t)(f0 + tl) * P.n + r) * nt; });
  __syncthreads();
  if (init_Tsrc) {  // f1plus = N_{-1} = T G_d   [PAPER.md:19, 67, 74]
    const float* zf = reinterpret_cast<const float*>(smem);
    for (int idx = threadIdx.x; idx < nf * nt; idx += blockDim.x) {
      const int tl = idx / nt, j = idx - tl * nt;
      init_Tsrc[((size_t)(f0 + tl) * P.n + r) * nt + j] = zf[2 * tl * MP + mkfft::padj((nt - j) & (nt - 1))];
    }
    __syncthreads();  // the in-place FFT below overwrites what this loop reads
  }
  fft_batch_fwd(smem, nf, MP, P.plan, P.tw);
  for (int idx = threadIdx.x; idx < P.nb * FT; idx += blockDim.x) {
    const int kk = idx / FT, tl = idx - kk * FT;
    if (tl >= nf) continue;
    float2 X = mkfft::rfft_bin(smem + tl * MP, P.plan, P.tw, P.klo + kk);
    if (conj_out) X.y = -X.y;  // spectrum of the time-reversed real trace
    Nhat[((size_t)kk * P.ld + r) * P.ldf + f0 + tl] = X;
  }
}

// ------------------------------------------------------------------------------------------------ k_inv
// grid (ceil(nfoc/FT), n); spec: [n][nb][ldf]; out[j] = sS*S[j] + sA*A[j] + sB*B[(nt-j)%nt]
__global__ void __launch_bounds__(kThreads) k_inv(const float2* __restrict__ spec, FftParams P, int FT, float* __restrict__ out,
                                                  float sS, const float* __restrict__ A, float sA,
                                                  const float* __restrict__ B, float sB) {
  extern __shared__ float2 smem[];
  const int MP = mkfft::padded_len(P.plan.M);
  const int r = blockIdx.y, f0 = blockIdx.x * FT;
  const int nf = min(FT, P.nfoc - f0);
  const int nt = P.plan.nt;
  const float2* srow = spec + (size_t)r * P.nb * P.ldf + f0;
  spectrum_to_Z<false>(smem, nf, FT, MP, P.plan, P.tw, P.klo, P.nb,
                       [&](int tl, int kk) { return __ldg(srow + (size_t)kk * P.ldf + tl); });
  __syncthreads();
  fft_batch_inv(smem, nf, MP, P.plan, P.tw);
  const float* zf = reinterpret_cast<const float*>(smem);
  for (int idx = threadIdx.x; idx < nf * nt; idx += blockDim.x) {
    const int tl = idx / nt, j = idx - tl * nt;
    const size_t base = ((size_t)(f0 + tl) * P.n + r) * nt;
    float v = sS * zf[2 * tl * MP + mkfft::padj(j)];
    if (A) v += sA * A[base + j];
    if (B) v += sB * B[base + ((nt - j) & (nt - 1))];
    out[base + j] = v;
  }
}

// ------------------------------------------------------------------------------------------------ k_post
// grid (ceil(nfoc/FT), n).  Shat, phat: [n][nb][ldf]; Nhat: [nb][ld][ldf]; h: [nfoc][n]; f1plus/f1min: [nfoc][n][nt]
__global__ void __launch_bounds__(kThreads) k_post(const float2* __restrict__ Shat, float2* __restrict__ phat, float2* __restrict__ Nhat,
                                                   const int* __restrict__ h, float* __restrict__ f1plus, float* __restrict__ f1min,
                                                   FftParams P, int FT, int parity_even, float* __restrict__ Ni_out) {
  extern __shared__ float2 smem[];
  const int MP = mkfft::padded_len(P.plan.M);
  const int r = blockIdx.y, f0 = blockIdx.x * FT;
  const int nf = min(FT, P.nfoc - f0);
  const int nt = P.plan.nt;
  const size_t rowoff = (size_t)r * P.nb * P.ldf + f0;
  // a3: p^ += S^ ; Z of conj(S^) so that the inverse transform yields u = T S directly  [PAPER.md:79, 71]
  spectrum_to_Z<true>(smem, nf, FT, MP, P.plan, P.tw, P.klo, P.nb, [&](int tl, int kk) {
    const size_t o = rowoff + (size_t)kk * P.ldf + tl;
    const float2 s = __ldg(Shat + o);
    float2 pv = phat[o];
    pv.x += s.x;
    pv.y += s.y;
    phat[o] = pv;
    return s;
  });
  __syncthreads();
  fft_batch_inv(smem, nf, MP, P.plan, P.tw);
  float* zf = reinterpret_cast<float*>(smem);
  // a5: N_i = -Theta u.  i even: f1min -= T N_i  <=>  f1min[j] += Theta[j] u[(nt-j)%nt];  i odd: f1plus += N_i
  //     [PAPER.md:82-85].  Only samples inside the window are touched.
  for (int idx = threadIdx.x; idx < nf * nt; idx += blockDim.x) {
    const int tl = idx / nt, j = idx - tl * nt;
    const int hh = h[(size_t)(f0 + tl) * P.n + r];
    if (j < hh || j > nt - hh) {
      const size_t o = ((size_t)(f0 + tl) * P.n + r) * nt + j;
      if (parity_even) f1min[o] += zf[2 * tl * MP + mkfft::padj((nt - j) & (nt - 1))];
      else f1plus[o] -= zf[2 * tl * MP + mkfft::padj(j)];
    }
  }
  __syncthreads();
  // a4: N_i in place (hard 0/1 window, strict inequality; G2)
  for (int idx = threadIdx.x; idx < nf * nt; idx += blockDim.x) {
    const int tl = idx / nt, j = idx - tl * nt;
    const int hh = h[(size_t)(f0 + tl) * P.n + r];
    const int a = 2 * tl * MP + mkfft::padj(j);
    const float v = (j < hh || j > nt - hh) ? -zf[a] : 0.f;
    zf[a] = v;
    if (Ni_out) Ni_out[((size_t)(f0 + tl) * P.n + r) * nt + j] = v;
  }
  __syncthreads();
  // a6: N^_i band
  fft_batch_fwd(smem, nf, MP, P.plan, P.tw);
  for (int idx = threadIdx.x; idx < P.nb * FT; idx += blockDim.x) {
    const int kk = idx / FT, tl = idx - kk * FT;
    if (tl >= nf) continue;
    Nhat[((size_t)kk * P.ld + r) * P.ldf + f0 + tl] = mkfft::rfft_bin(smem + tl * MP, P.plan, P.tw, P.klo + kk);
  }
}

int pick_ft(const mk_ctx* c, int nfoc, int cap) {
  const size_t per = (size_t)mkfft::padded_len(c->plan.M) * sizeof(float2);
  int ft = (int)(72000 / per);
  if (ft < 1) ft = 1;
  if (ft > cap) ft = cap;
  if (ft > nfoc) ft = nfoc;
  return ft;
}

FftParams make_params(const mk_ctx* c, int nfoc, int ldf) {
  FftParams P;
  P.plan = c->plan;
  P.tw = c->d_tw;
  P.n = c->n;
  P.nb = c->nb;
  P.klo = c->klo;
  P.ld = c->ld;
  P.ldf = ldf;
  P.nfoc = nfoc;
  return P;
}

template <typename K>
int set_smem(mk_ctx* c, K kernel, size_t bytes) {
  if (bytes > c->smem_optin) return set_err(c, MK_ERR_INVALID_ARG, "trace too long for shared memory");
  return check_cuda(c, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes), "cudaFuncSetAttribute");
}

}  // namespace

int launch_window(mk_ctx* c, const float* d_td, int* d_h, int ntr) {
  k_window<<<(ntr + 255) / 256, 256, 0, c->stream>>>(d_td, d_h, ntr, c->dt, c->eps, c->nt);
  ++c->launches;
  return check_cuda(c, cudaGetLastError(), "k_window");
}

int launch_load_R(mk_ctx* c, const float* d_R_time, int shot0, int nshots) {
  const int ST = pick_ft(c, nshots, 8);
  const size_t smem = (size_t)ST * mkfft::padded_len(c->plan.M) * sizeof(float2);
  if (int rc = set_smem(c, k_load_R, smem)) return rc;
  const dim3 grid((nshots + ST - 1) / ST, c->n);
  const float sm = (float)(c->dt * c->dx), se = (float)(c->dt * c->dx * 0.5);
  k_load_R<<<grid, kThreads, smem, c->stream>>>(d_R_time, c->d_Rhat, make_params(c, 0, 0), shot0, nshots, ST, sm, se);
  ++c->launches;
  return check_cuda(c, cudaGetLastError(), "k_load_R");
}

int launch_fwd(mk_ctx* c, const float* d_src, float2* d_Nhat, int nfoc, int ldf, bool conj_out, float* d_init_Tsrc) {
  const int FT = pick_ft(c, nfoc, 8);
  const size_t smem = (size_t)FT * mkfft::padded_len(c->plan.M) * sizeof(float2);
  if (int rc = set_smem(c, k_fwd, smem)) return rc;
  const dim3 grid((nfoc + FT - 1) / FT, c->n);
  k_fwd<<<grid, kThreads, smem, c->stream>>>(d_src, d_Nhat, make_params(c, nfoc, ldf), FT, conj_out ? 1 : 0, d_init_Tsrc);
  ++c->launches;
  return check_cuda(c, cudaGetLastError(), "k_fwd");
}

int launch_inv(mk_ctx* c, const float2* d_spec, int nfoc, int ldf, float* d_out, float sS, const float* d_A, float sA,
               const float* d_B, float sB) {
  const int FT = pick_ft(c, nfoc, 8);
  const size_t smem = (size_t)FT * mkfft::padded_len(c->plan.M) * sizeof(float2);
  if (int rc = set_smem(c, k_inv, smem)) return rc;
  const dim3 grid((nfoc + FT - 1) / FT, c->n);
  k_inv<<<grid, kThreads, smem, c->stream>>>(d_spec, make_params(c, nfoc, ldf), FT, d_out, sS, d_A, sA, d_B, sB);
  ++c->launches;
  return check_cuda(c, cudaGetLastError(), "k_inv");
}

int launch_post(mk_ctx* c, int parity_even, float* d_Ni_out) {
  const int FT = pick_ft(c, c->nfoc, 8);
  const size_t smem = (size_t)FT * mkfft::padded_len(c->plan.M) * sizeof(float2);
  if (int rc = set_smem(c, k_post, smem)) return rc;
  const dim3 grid((c->nfoc + FT - 1) / FT, c->n);
  k_post<<<grid, kThreads, smem, c->stream>>>(c->d_Shat, c->d_phat, c->d_Nhat, c->d_h, c->d_f1plus, c->d_f1min,
                                              make_params(c, c->nfoc, c->ldf), FT, parity_even, d_Ni_out);
  ++c->launches;
  return check_cuda(c, cudaGetLastError(), "k_post");
}

}  // namespace mk

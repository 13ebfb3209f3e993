// fft_core.cuh — in-shared-memory real FFT building blocks for traces of nt = 2M samples (nt a power of two).
//
// A real trace x[0..nt) is viewed in place as M complex numbers z[m] = x[2m] + i x[2m+1]; one complex FFT of
// length M plus an O(M) split step gives the half spectrum X[0..M] (reading G11: forward e^{-2 pi i k j / nt},
// the inverse carries 1/nt).  The complex FFT is an in-place decimation-in-frequency pass sequence (radix 8,
// finished by one radix 4 or 2 pass), which leaves the spectrum in digit-reversed order; the inverse is the
// exact mirror (decimation in time from digit-reversed input), so no reordering pass is ever run: the split
// steps address Z[k] through freq_pos(k).
//
// Everything here is written per butterfly index so that the CUDA kernels call it as
//   for (b = tid; b < ntraces * M/r; b += nthreads) pass(...);  __syncthreads();
// The functions are plain C++ (MK_HD), so the index arithmetic can also be exercised on the host.
#pragma once

#ifdef __CUDACC__
#define MK_HD __host__ __device__ __forceinline__
#else
#include <cmath>
#define MK_HD inline
struct float2 {
  float x, y;
};
static inline float2 make_float2(float x, float y) { return float2{x, y}; }
#endif

namespace mkfft {

constexpr int kMaxPass = 6;

struct Plan {
  int nt;    // real trace length
  int M;     // complex length nt/2
  int logM;
  int npass;
  int lgr[kMaxPass];  // log2(radix) of forward pass p
  int lgL[kMaxPass];  // log2(block length) of forward pass p
};

inline Plan make_plan(int nt) {
  Plan p{};
  p.nt = nt;
  p.M = nt / 2;
  p.logM = 0;
  while ((1 << p.logM) < p.M) ++p.logM;
  int left = p.logM, np = 0;
  while (left > 0) {
    const int l = left >= 3 && left != 4 ? 3 : (left >= 2 ? 2 : 1);  // 8,8,...,then 4,4 / 4 / 2
    p.lgr[np] = l;
    p.lgL[np] = left;
    left -= l;
    ++np;
  }
  p.npass = np;
  return p;
}

// shared-memory index padding: one complex of padding per 16 keeps every pass at <= 2-way bank conflicts
MK_HD int padi(int i) { return i + (i >> 4); }
MK_HD int padded_len(int M) { return M + (M >> 4) + 1; }
// float (real-sample) index j of the trace -> float index inside the padded complex buffer
MK_HD int padj(int j) { return 2 * padi(j >> 1) + (j & 1); }

MK_HD float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
MK_HD float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
MK_HD float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
MK_HD float2 cmulc(float2 a, float2 b) { return make_float2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }  // a*conj(b)

// position of frequency k (0 <= k < M) after the forward passes
MK_HD int freq_pos(const Plan& p, int k) {
  int pos = 0, lg = p.logM;
  for (int i = 0; i < p.npass; ++i) {
    const int l = p.lgr[i];
    lg -= l;
    pos += (k & ((1 << l) - 1)) << lg;
    k >>= l;
  }
  return pos;
}

// ---- small DFTs in registers; INV = false: e^{-2 pi i jm/R}, INV = true: e^{+2 pi i jm/R}
template <bool INV>
MK_HD float2 mul_mi(float2 a) {  // a * (-i) forward, a * (+i) inverse
  return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
}

template <bool INV>
MK_HD void dft2(float2& a0, float2& a1) {
  const float2 t = a0;
  a0 = cadd(t, a1);
  a1 = csub(t, a1);
}

template <bool INV>
MK_HD void dft4(float2& a0, float2& a1, float2& a2, float2& a3) {
  const float2 t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), t3 = mul_mi<INV>(csub(a1, a3));
  a0 = cadd(t0, t2);
  a2 = csub(t0, t2);
  a1 = cadd(t1, t3);
  a3 = csub(t1, t3);
}

template <bool INV>
MK_HD void dft8(float2* a) {
  dft4<INV>(a[0], a[2], a[4], a[6]);  // E_m in a[0], a[2], a[4], a[6]
  dft4<INV>(a[1], a[3], a[5], a[7]);  // O_m in a[1], a[3], a[5], a[7]
  const float c = 0.70710678118654752440f;
  // omega_8^m O_m
  const float2 o0 = a[1];
  const float2 o1 = INV ? make_float2(c * (a[3].x - a[3].y), c * (a[3].x + a[3].y))
                        : make_float2(c * (a[3].x + a[3].y), c * (a[3].y - a[3].x));
  const float2 o2 = mul_mi<INV>(a[5]);
  const float2 o3 = INV ? make_float2(-c * (a[7].x + a[7].y), c * (a[7].x - a[7].y))
                        : make_float2(c * (a[7].y - a[7].x), -c * (a[7].x + a[7].y));
  const float2 e0 = a[0], e1 = a[2], e2 = a[4], e3 = a[6];
  a[0] = cadd(e0, o0);
  a[4] = csub(e0, o0);
  a[1] = cadd(e1, o1);
  a[5] = csub(e1, o1);
  a[2] = cadd(e2, o2);
  a[6] = csub(e2, o2);
  a[3] = cadd(e3, o3);
  a[7] = csub(e3, o3);
}

template <int LGR, bool INV>
MK_HD void dft_small(float2* a) {
  if (LGR == 3) dft8<INV>(a);
  else if (LGR == 2) dft4<INV>(a[0], a[1], a[2], a[3]);
  else dft2<INV>(a[0], a[1]);
}

// Twiddles w[m] = tw[m * tstep], m = 1 .. R-1.  Only the power-of-two multiples are read from the table (the table
// lives in global memory / L1); the others are products of two table entries (one extra rounding, ~6e-8).
template <int LGR>
MK_HD void load_twiddles(float2* w, const float2* __restrict__ tw, int tstep) {
  w[0] = make_float2(1.f, 0.f);
  w[1] = tw[tstep];
  if constexpr (LGR >= 2) {
    w[2] = tw[2 * tstep];
    w[3] = cmul(w[1], w[2]);
  }
  if constexpr (LGR >= 3) {
    w[4] = tw[4 * tstep];
    w[5] = cmul(w[4], w[1]);
    w[6] = cmul(w[4], w[2]);
    w[7] = cmul(w[4], w[3]);
  }
}

// One butterfly (index t in [0, M >> LGR)) of forward pass with block length 2^lgL.  z: padded trace buffer,
// tw[k] = e^{-2 pi i k / nt}, k in [0, nt).
template <int LGR>
MK_HD void fwd_butterfly(float2* z, const float2* __restrict__ tw, int nt, int lgL, int t) {
  constexpr int R = 1 << LGR;
  const int lgq = lgL - LGR;
  const int blk = t >> lgq, i = t & ((1 << lgq) - 1);
  const int base = (blk << lgL) + i;
  float2 a[R];
#pragma unroll
  for (int j = 0; j < R; ++j) a[j] = z[padi(base + (j << lgq))];
  dft_small<LGR, false>(a);
  const int tstep = i * (nt >> lgL);  // w_L^{i m} = tw[i m nt/L]
  float2 w[R];
  load_twiddles<LGR>(w, tw, tstep);
#pragma unroll
  for (int m = 1; m < R; ++m) a[m] = cmul(a[m], w[m]);
#pragma unroll
  for (int m = 0; m < R; ++m) z[padi(base + (m << lgq))] = a[m];
}

// Mirror of fwd_butterfly: conj twiddles first, then the conjugate small DFT.
template <int LGR>
MK_HD void inv_butterfly(float2* z, const float2* __restrict__ tw, int nt, int lgL, int t) {
  constexpr int R = 1 << LGR;
  const int lgq = lgL - LGR;
  const int blk = t >> lgq, i = t & ((1 << lgq) - 1);
  const int base = (blk << lgL) + i;
  float2 a[R];
#pragma unroll
  for (int m = 0; m < R; ++m) a[m] = z[padi(base + (m << lgq))];
  const int tstep = i * (nt >> lgL);
  float2 w[R];
  load_twiddles<LGR>(w, tw, tstep);
#pragma unroll
  for (int m = 1; m < R; ++m) a[m] = cmulc(a[m], w[m]);
  dft_small<LGR, true>(a);
#pragma unroll
  for (int j = 0; j < R; ++j) z[padi(base + (j << lgq))] = a[j];
}

// ---- 32-point DFT held entirely in registers (the building block of the register-resident path, mk_fft_fast.cu):
// 32 = 4 x 8, natural order in and out; every index below is a compile-time constant after unrolling, so the
// twiddles are immediates and the final reordering is a renaming of registers.
MK_HD float w32_cos(int m) {
  constexpr float t[32] = {1.f, 0.980785251f, 0.923879504f, 0.831469595f, 0.707106769f, 0.555570245f, 0.382683426f, 0.195090324f,
                           0.f, -0.195090324f, -0.382683426f, -0.555570245f, -0.707106769f, -0.831469595f, -0.923879504f, -0.980785251f,
                           -1.f, -0.980785251f, -0.923879504f, -0.831469595f, -0.707106769f, -0.555570245f, -0.382683426f, -0.195090324f,
                           0.f, 0.195090324f, 0.382683426f, 0.555570245f, 0.707106769f, 0.831469595f, 0.923879504f, 0.980785251f};
  return t[m & 31];
}
MK_HD float w32_sin(int m) { return w32_cos(m - 8); }  // sin(x) = cos(x - pi/2)

template <bool INV>
MK_HD void fft32(float2 (&a)[32]) {
  // input n = 8 n1 + n2, output k = k1 + 4 k2
#pragma unroll
  for (int n2 = 0; n2 < 8; ++n2) dft4<INV>(a[n2], a[8 + n2], a[16 + n2], a[24 + n2]);  // a[8 k1 + n2] = Y[k1][n2]
#pragma unroll
  for (int k1 = 1; k1 < 4; ++k1)
#pragma unroll
    for (int n2 = 1; n2 < 8; ++n2) {
      const float2 w = make_float2(w32_cos(k1 * n2), -w32_sin(k1 * n2));  // e^{-2 pi i k1 n2 / 32}
      a[8 * k1 + n2] = INV ? cmulc(a[8 * k1 + n2], w) : cmul(a[8 * k1 + n2], w);
    }
#pragma unroll
  for (int k1 = 0; k1 < 4; ++k1) dft8<INV>(&a[8 * k1]);  // a[8 k1 + k2] = X[k1 + 4 k2]
  float2 b[32];
#pragma unroll
  for (int k1 = 0; k1 < 4; ++k1)
#pragma unroll
    for (int k2 = 0; k2 < 8; ++k2) b[k1 + 4 * k2] = a[8 * k1 + k2];
#pragma unroll
  for (int i = 0; i < 32; ++i) a[i] = b[i];
}

// ---- real <-> half-spectrum split steps
// Forward: X[k] (0 <= k <= M) of the real trace from the digit-reversed Z held in z.
MK_HD float2 rfft_bin(const float2* z, const Plan& p, const float2* __restrict__ tw, int k) {
  const int M = p.M;
  const float2 a = z[padi(freq_pos(p, k & (M - 1)))];
  const float2 b = z[padi(freq_pos(p, (M - k) & (M - 1)))];
  const float er = 0.5f * (a.x + b.x), ei = 0.5f * (a.y - b.y);   // E = (a + conj b)/2
  const float orr = 0.5f * (a.y + b.y), oi = -0.5f * (a.x - b.x);  // O = (a - conj b)/(2i)
  const float2 w = tw[k];
  return make_float2(er + w.x * orr - w.y * oi, ei + w.x * oi + w.y * orr);
}

// Inverse: Z[k] (0 <= k < M), already scaled by `scale`, from X[k] and X[M-k]; twk = tw[k].
MK_HD float2 irfft_pre(float2 Xk, float2 Xmk, float2 twk, float scale) {
  const float er = Xk.x + Xmk.x, ei = Xk.y - Xmk.y;  // X[k] + conj X[M-k]
  const float dr = Xk.x - Xmk.x, di = Xk.y + Xmk.y;  // X[k] - conj X[M-k]
  // O2 = (dr + i di) * conj(tw) ; Z = (E2 + i O2) * scale   (the 1/2 of E and O is folded into scale)
  const float o_r = dr * twk.x + di * twk.y, o_i = di * twk.x - dr * twk.y;
  return make_float2(scale * (er - o_i), scale * (ei + o_r));
}

}  // namespace mkfft

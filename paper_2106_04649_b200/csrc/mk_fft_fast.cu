// mk_fft_fast.cu — register-resident transform kernels for nt = 2048 and nt = 4096 (every BASELINE.json config but
// the tiny one): the same four per-trace kernels as mk_fft_kernels.cu, built on
// a 1024-point complex FFT that ONE WARP runs with 32 values per thread:
//
//   four-step FFT, 1024 = 32 x 32:  a 32-point DFT in registers (fft_core.cuh fft32), the middle twiddles W_1024^{k1 t}
//   from a 32 x 32 table, ONE transposition through shared memory (rows padded to 33, conflict-free both ways), and a
//   second 32-point DFT in registers.  Input: lane t holds x[t + 32 q], q = 0..31; output: lane t holds X[t + 32 q].
//   The transform of the time-domain result therefore starts straight from the registers the window left.
//
// A real trace of nt samples is M = nt/2 complex numbers z[m] = x[2m] + i x[2m+1] (fft_core.cuh).  nt = 2048: M = 1024,
// one warp per trace.  nt = 4096: M = 2048 = 2 x 1024, two warps per trace (HF = 2): warp h owns the samples
// z[2 n' + h]; the radix-2 step that joins the two halves is folded into the shared-memory phases that exist anyway
// (decimation in frequency on the way in: A_h[k] = (Z[k] + (-1)^h Z[k + 1024]) W_2048^{-h k}; decimation in time on
// the way out: Z[k] = F_0[k mod 1024] +- W_2048^{k mod 1024} F_1[k mod 1024]).
//
// One CTA = one receiver r and FT consecutive focal points (the S^[r][k][f..] reads and N^[k][r][f..] writes are
// contiguous 8 FT-byte segments); its phases:
//   P1 (CTA-wide, focal point fastest)  half spectra from HBM -> Z in shared memory (p^ += S^ on the way)
//   P2 (per warp)  inverse transform, registers <- time samples
//   P3 (per warp)  window, accumulation into f1min / f1plus straight from registers (coalesced float2 rows)
//   P4 (per warp)  forward transform, Z -> shared memory
//   P5 (CTA-wide)  band of the half spectrum -> operand of the next contraction
// Compared with the generic kernels this is ~8 shared-memory accesses per complex element and pass instead of ~21,
// no digit-reversal arithmetic, and warp-level synchronisation only inside P2..P4.
#include "mk_fft_common.cuh"

namespace mk {

namespace {

using mkfft::cadd;
using mkfft::cmul;
using mkfft::cmulc;
using mkfft::csub;

constexpr int SUB = 32 * 33;  // float2 per 1024-point block: 32 rows of 32 + 1 pad

// Accumulations into global memory (p^ += S^, f1min += w, f1plus -= w) are reductions performed by the L2: every address is
// touched once per launch, so the result is the same round-to-nearest sum a load / add / store would give (subnormals are
// flushed), but no thread ever waits for the old value — the pass has ONE exposed global round trip left (the S^ loads)
__device__ __forceinline__ void red_add2(float* p, float a, float b) {
  asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(a), "f"(b) : "memory");
}
__device__ __forceinline__ void red_add4(float2* p, float4 v) {
  asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

template <int HF>
struct Geo {
  static constexpr int M = 1024 * HF;      // complex length of a trace
  static constexpr int TS = HF * SUB + 2;  // float2 between traces in shared memory (== 2 mod 16: P1 / P5 conflict-free)
};

struct FastParams {
  const float2* tw;    // [nt]      e^{-2 pi i k / nt}
  const float* wscale; // [ns]     dt * w[s] (k_load_R_fast)
  const float2* tw1k;  // [32][32]  e^{-2 pi i k1 t / 1024}
  int nt, n, nb, klo, ld, ldf, nfoc;
  int tiled;  // k_load_R_fast: layout of R^ (rhat_index)
  int r0;  // first receiver row of this context (row sharding): grid row b handles receiver r0 + b
  int warm;  // warm_tables (off with MK_OPT_TUNE bit 13)
};

// natural index k (0 <= k < M) of Z -> float2 offset inside the trace's shared-memory block
__device__ __forceinline__ int zaddr(int k) { return (k >> 10) * SUB + ((k & 1023) >> 5) * 33 + (k & 31); }

// all warps of one trace (HF = 1: the warp itself)
template <int HF>
__device__ __forceinline__ void trace_sync(int tl) {
  if (HF == 1) {
    __syncwarp();
  } else {  // named barriers 1..8 (immediate ids, so that only these are reserved); FT <= 8
    switch (tl) {
      case 0: asm volatile("bar.sync 1, %0;" ::"n"(32 * HF) : "memory"); break;
      case 1: asm volatile("bar.sync 2, %0;" ::"n"(32 * HF) : "memory"); break;
      case 2: asm volatile("bar.sync 3, %0;" ::"n"(32 * HF) : "memory"); break;
      case 3: asm volatile("bar.sync 4, %0;" ::"n"(32 * HF) : "memory"); break;
      case 4: asm volatile("bar.sync 5, %0;" ::"n"(32 * HF) : "memory"); break;
      case 5: asm volatile("bar.sync 6, %0;" ::"n"(32 * HF) : "memory"); break;
      case 6: asm volatile("bar.sync 7, %0;" ::"n"(32 * HF) : "memory"); break;
      default: asm volatile("bar.sync 8, %0;" ::"n"(32 * HF) : "memory"); break;
    }
  }
}

// Few traces (every CTA of the launch resident at once: the kernel is one latency chain per warp): the twiddle tables, written
// once at mk_create, are pulled into this SM's L1 while the kernel in front is still draining (before pdl_wait; constant
// data only: anything a kernel of the run writes may still be in flight there).
__device__ __forceinline__ void warm_tables(const FastParams& P, bool on) {
  if (!on || gridDim.x * gridDim.y > 2048u) return;
  const float4* t1 = reinterpret_cast<const float4*>(P.tw1k);
  for (int i = threadIdx.x; i < 512; i += blockDim.x) {
    const float4 v = __ldg(t1 + i);
    asm volatile("" ::"f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w));
  }
  const float4* t2 = reinterpret_cast<const float4*>(P.tw + (P.klo & ~1));
  for (int i = threadIdx.x; i < (P.nb + 3) / 2; i += blockDim.x) {
    const float4 v = __ldg(t2 + i);
    asm volatile("" ::"f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w));
  }
}

// 1024-point complex FFT by one warp.  In: lane t holds a[q] = x[t + 32 q].  Out: lane t holds a[q] = X[t + 32 q].
// scratch: 1056 float2 owned by this warp (contents destroyed).  INV: e^{+...}, no scaling.
template <bool INV>
__device__ __forceinline__ void warp_fft1024(float2 (&a)[32], float2* scratch, const float2* __restrict__ tw1k, int t) {
  mkfft::fft32<INV>(a);  // a[k1] = Y[k1][n2 = t]
#pragma unroll
  for (int k1 = 1; k1 < 32; ++k1) {
    const float2 w = __ldg(tw1k + k1 * 32 + t);
    a[k1] = INV ? cmulc(a[k1], w) : cmul(a[k1], w);
  }
  __syncwarp();  // every lane is done reading the scratch block
#pragma unroll
  for (int k1 = 0; k1 < 32; ++k1) scratch[k1 * 33 + t] = a[k1];
  __syncwarp();
#pragma unroll
  for (int n2 = 0; n2 < 32; ++n2) a[n2] = scratch[t * 33 + n2];
  mkfft::fft32<INV>(a);  // a[k2] = X[k1 = t + 32 k2]
}

// P2 load: this warp's input of the inverse transform from the natural-order Z in shared memory
template <int HF>
__device__ __forceinline__ void load_Z(float2 (&a)[32], const float2* zt, int hf, int t, const float2* __restrict__ tw) {
  if (HF == 1) {
#pragma unroll
    for (int n1 = 0; n1 < 32; ++n1) a[n1] = zt[n1 * 33 + t];
  } else {
#pragma unroll
    for (int n1 = 0; n1 < 32; ++n1) {
      const float2 z0 = zt[n1 * 33 + t], z1 = zt[SUB + n1 * 33 + t];
      if (hf == 0) a[n1] = cadd(z0, z1);
      else a[n1] = cmulc(csub(z0, z1), __ldg(tw + 2 * (32 * n1 + t)));  // e^{+2 pi i k / 2048} = conj tw[2k], nt = 4096
    }
  }
}

// P4 store: this warp's forward result -> natural-order blocks in shared memory (HF = 2: the odd half pre-twiddled)
template <int HF>
__device__ __forceinline__ void store_Z(const float2 (&a)[32], float2* zt, int hf, int t, const float2* __restrict__ tw) {
  __syncwarp();
#pragma unroll
  for (int k2 = 0; k2 < 32; ++k2) {
    float2 v = a[k2];
    if (HF == 2 && hf == 1) v = cmul(v, __ldg(tw + 2 * (t + 32 * k2)));
    zt[hf * SUB + k2 * 33 + t] = v;
  }
}

template <int HF>
__device__ __forceinline__ float2 Zval(const float2* zt, int k) {  // Z[k], 0 <= k < M, after store_Z
  if (HF == 1) return zt[zaddr(k)];
  const int kp = k & 1023, ad = (kp >> 5) * 33 + (kp & 31);
  const float2 e = zt[ad], o = zt[SUB + ad];
  return k < 1024 ? cadd(e, o) : csub(e, o);
}

// X[k] (0 <= k <= M) of the real trace from its Z (same arithmetic as mkfft::rfft_bin)
template <int HF>
__device__ __forceinline__ float2 rfft_bin_fast(const float2* zt, const float2* __restrict__ tw, int k) {
  constexpr int M = Geo<HF>::M;
  const float2 a = Zval<HF>(zt, k & (M - 1));
  const float2 b = Zval<HF>(zt, (M - k) & (M - 1));
  const float er = 0.5f * (a.x + b.x), ei = 0.5f * (a.y - b.y);
  const float orr = 0.5f * (a.y + b.y), oi = -0.5f * (a.x - b.x);
  const float2 w = __ldg(tw + k);
  return make_float2(er + w.x * orr - w.y * oi, ei + w.x * oi + w.y * orr);
}

// P1.  Z (natural order, scaled by 1/nt) of all FT traces from their band-limited half spectra.  CTA-wide: consecutive
// threads take consecutive focal points of one bin.  load(tl, kk, aux) returns X[klo + kk] of trace tl (and may fetch
// a side value into aux); commit(tl, kk, X, aux) runs afterwards.  Both are called exactly once per in-band (k, tl);
// the loads of four items are issued before anything is consumed.  CONJ: transform conj(X) instead (time reversal).
template <int HF, typename Load, typename Commit>
__device__ __forceinline__ void spectrum_in(float2* smem, int nf, int lgFT, bool conj_in, const FastParams& P, Load load,
                                            Commit commit) {
  constexpr int M = Geo<HF>::M, half = M >> 1, TS = Geo<HF>::TS;
  const int FT = 1 << lgFT, nthr = blockDim.x;
  const float scale = 1.0f / (2.0f * (float)M);
  const int total = (half + 1) << lgFT;
  const int klo = P.klo, khi1 = P.klo + P.nb;
  constexpr int kBatch = 8;
  for (int i0 = threadIdx.x; i0 < total; i0 += kBatch * nthr) {
    float2 a[kBatch], b[kBatch], xa[kBatch], xb[kBatch];
#pragma unroll
    for (int u = 0; u < kBatch; ++u) {
      const int idx = i0 + u * nthr;
      a[u] = b[u] = xa[u] = xb[u] = make_float2(0.f, 0.f);
      if (idx < total) {
        const int k = idx >> lgFT, tl = idx & (FT - 1), k2 = M - k;
        if (tl < nf) {
          if (k >= klo && k < khi1) a[u] = load(tl, k - klo, xa[u]);
          if (k2 != k && k2 >= klo && k2 < khi1) b[u] = load(tl, k2 - klo, xb[u]);
        }
      }
    }
#pragma unroll
    for (int u = 0; u < kBatch; ++u) {
      const int idx = i0 + u * nthr;
      if (idx >= total) continue;
      const int k = idx >> lgFT, tl = idx & (FT - 1), k2 = M - k;
      if (tl >= nf) continue;
      if (k >= klo && k < khi1) commit(tl, k - klo, a[u], xa[u]);
      if (k2 != k && k2 >= klo && k2 < khi1) commit(tl, k2 - klo, b[u], xb[u]);
      float2 x = a[u], y = b[u];
      if (k2 == k) y = x;
      if (k == 0) {  // DC and Nyquist are real for a real trace (irfft convention)
        x.y = 0.f;
        y.y = 0.f;
      }
      if (conj_in) {
        x.y = -x.y;
        y.y = -y.y;
      }
      float2* zt = smem + tl * TS;
      zt[zaddr(k)] = mkfft::irfft_pre(x, y, __ldg(P.tw + k), scale);
      if (k2 < M && k2 != k) zt[zaddr(k2)] = mkfft::irfft_pre(y, x, __ldg(P.tw + k2), scale);
    }
  }
}

// P5.  emit(tl, kk, X[klo + kk]) for every in-band bin of every trace; CTA-wide, trace index fastest
template <int HF, typename Emit>
__device__ __forceinline__ void band_out(const float2* smem, int nf, int lgFT, const FastParams& P, Emit emit) {
  constexpr int TS = Geo<HF>::TS, kBatch = 4;
  const int FT = 1 << lgFT, total = P.nb << lgFT, nthr = blockDim.x;
  for (int i0 = threadIdx.x; i0 < total; i0 += kBatch * nthr) {
    float2 X[kBatch];
#pragma unroll
    for (int u = 0; u < kBatch; ++u) {  // shared-memory and twiddle loads of the whole batch first
      const int idx = i0 + u * nthr;
      if (idx < total && (idx & (FT - 1)) < nf) X[u] = rfft_bin_fast<HF>(smem + (idx & (FT - 1)) * TS, P.tw, P.klo + (idx >> lgFT));
    }
#pragma unroll
    for (int u = 0; u < kBatch; ++u) {
      const int idx = i0 + u * nthr;
      if (idx < total && (idx & (FT - 1)) < nf) emit(idx & (FT - 1), idx >> lgFT, X[u]);
    }
  }
}

// float offset inside a trace of the sample pair held in register q of lane t of warp hf
template <int HF>
__device__ __forceinline__ int sample_j(int q, int t, int hf) { return 2 * (HF * (t + 32 * q) + hf); }

struct Who {
  int tl, hf, t;
};
template <int HF>
__device__ __forceinline__ Who who() {
  const int w = threadIdx.x >> 5;
  return Who{w / HF, w % HF, (int)(threadIdx.x & 31)};
}

// P3 load of a whole trace: lane t, register q <- samples (j, j+1), j = sample_j(q)
template <int HF>
__device__ __forceinline__ void load_time(float2 (&a)[32], const float* __restrict__ src, const Who& me) {
#pragma unroll
  for (int q = 0; q < 32; ++q) a[q] = __ldg(reinterpret_cast<const float2*>(src + sample_j<HF>(q, me.t, me.hf)));
}


// ---- P1 / P5 with two focal points per thread (FT = 4 or 8, even ldf): 128-bit accesses of S^, p^ and the operand.
// P1 needs the usual band shape 1 <= klo, khi < M/2 (no DC / Nyquist / mid bin, the mirror M - k of an in-band bin is
// out of band): then Z[k] and Z[M-k] depend on X[k] alone,
//   o = X tw*,  Z[k] = s (X.x - o.y, X.y + o.x),  Z[M-k] = s (X.x + o.y, o.x - X.y)      (irfft_pre with the other bin 0,
//   tw[M-k] = -conj tw[k]), and every other Z is zero.  All loads of a thread are issued before anything is consumed.
__device__ __forceinline__ bool simple_band(const FastParams& P, int M) { return P.klo >= 1 && P.klo + P.nb - 1 < M / 2; }

template <int HF, bool RMW>
__device__ __forceinline__ void spectrum_in_pairs(float2* smem, int nf, int lgFT, bool conj_in, const FastParams& P,
                                                  const float2* __restrict__ Srow, float2* prow) {
  constexpr int M = Geo<HF>::M, TS = Geo<HF>::TS, kBatch = 8 / HF;
  const int nthr = blockDim.x, klo = P.klo, khi = P.klo + P.nb - 1;
  const float scale = 1.0f / (2.0f * (float)M);
  {  // zero fill of the out-of-band Z: k in [0, klo) u (khi, M - khi) u (M - klo, M)
    const int n0 = klo, n1 = M - 2 * khi - 1, nz = n0 + n1 + (klo - 1);
    for (int idx = threadIdx.x; idx < (nz << lgFT); idx += nthr) {
      const int tl = idx & ((1 << lgFT) - 1), j = idx >> lgFT;
      const int k = j < n0 ? j : (j < n0 + n1 ? khi + 1 + (j - n0) : M - klo + 1 + (j - n0 - n1));
      if (tl < nf) smem[tl * TS + zaddr(k)] = make_float2(0.f, 0.f);
    }
  }
  const int lgP = lgFT - 1, pm = (1 << lgP) - 1;  // focal-point pairs per bin
  const int total = P.nb << lgP;
  for (int i0 = threadIdx.x; i0 < total; i0 += kBatch * nthr) {
    float4 sv[kBatch];
#pragma unroll
    for (int u = 0; u < kBatch; ++u) {
      const int idx = i0 + u * nthr;
      if (idx < total && 2 * (idx & pm) < nf) {
        const size_t o = (size_t)(idx >> lgP) * P.ldf + 2 * (idx & pm);
        sv[u] = __ldg(reinterpret_cast<const float4*>(Srow + o));
      }
    }
#pragma unroll
    for (int u = 0; u < kBatch; ++u) {
      const int idx = i0 + u * nthr;
      if (idx >= total) continue;
      const int kk = idx >> lgP, t0 = 2 * (idx & pm), k = klo + kk;
      if (t0 >= nf) continue;
      if (RMW) red_add4(prow + (size_t)kk * P.ldf + t0, sv[u]);
      const float2 tw = __ldg(P.tw + k);
      const int a0 = zaddr(k), a1 = zaddr(M - k);
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        if (t0 + e >= nf) continue;
        const float xr = e ? sv[u].z : sv[u].x, xi0 = e ? sv[u].w : sv[u].y;
        const float xi = conj_in ? -xi0 : xi0;
        const float o_r = xr * tw.x + xi * tw.y, o_i = xi * tw.x - xr * tw.y;
        float2* zt = smem + (t0 + e) * TS;
        zt[a0] = make_float2(scale * (xr - o_i), scale * (xi + o_r));
        zt[a1] = make_float2(scale * (xr + o_i), scale * (o_r - xi));
      }
    }
  }
}


// The same for any FT with one focal point per thread (single-focal runs: FT = 1, S^ contiguous in the bin index)
template <int HF, bool RMW>
__device__ __forceinline__ void spectrum_in_singles(float2* smem, int nf, int lgFT, bool conj_in, const FastParams& P,
                                                    const float2* __restrict__ Srow, float2* prow) {
  constexpr int M = Geo<HF>::M, TS = Geo<HF>::TS, kBatch = 8;
  const int nthr = blockDim.x, klo = P.klo, khi = P.klo + P.nb - 1, fm = (1 << lgFT) - 1;
  const float scale = 1.0f / (2.0f * (float)M);
  {
    const int n0 = klo, n1 = M - 2 * khi - 1, nz = n0 + n1 + (klo - 1);
    for (int idx = threadIdx.x; idx < (nz << lgFT); idx += nthr) {
      const int tl = idx & fm, j = idx >> lgFT;
      const int k = j < n0 ? j : (j < n0 + n1 ? khi + 1 + (j - n0) : M - klo + 1 + (j - n0 - n1));
      if (tl < nf) smem[tl * TS + zaddr(k)] = make_float2(0.f, 0.f);
    }
  }
  const int total = P.nb << lgFT;
  for (int i0 = threadIdx.x; i0 < total; i0 += kBatch * nthr) {
    float2 sv[kBatch], tw[kBatch];
#pragma unroll
    for (int u = 0; u < kBatch; ++u) {
      const int idx = i0 + u * nthr;
      if (idx < total && (idx & fm) < nf) {
        const size_t o = (size_t)(idx >> lgFT) * P.ldf + (idx & fm);
        sv[u] = __ldg(Srow + o);
        tw[u] = __ldg(P.tw + klo + (idx >> lgFT));
      }
    }
#pragma unroll
    for (int u = 0; u < kBatch; ++u) {
      const int idx = i0 + u * nthr;
      if (idx >= total || (idx & fm) >= nf) continue;
      const int kk = idx >> lgFT, tl = idx & fm, k = klo + kk;
      if (RMW) red_add2(reinterpret_cast<float*>(prow + (size_t)kk * P.ldf + tl), sv[u].x, sv[u].y);
      const float xr = sv[u].x, xi = conj_in ? -sv[u].y : sv[u].y;
      const float o_r = xr * tw[u].x + xi * tw[u].y, o_i = xi * tw[u].x - xr * tw[u].y;
      float2* zt = smem + tl * TS;
      zt[zaddr(k)] = make_float2(scale * (xr - o_i), scale * (xi + o_r));
      zt[zaddr(M - k)] = make_float2(scale * (xr + o_i), scale * (o_r - xi));
    }
  }
}

// P5: emit2(kk, first trace t0 (even), X of t0, X of t0 + 1 (zero if that trace does not exist), whether it exists)
template <int HF, typename Emit2>
__device__ __forceinline__ void band_out_pairs(const float2* smem, int nf, int lgFT, const FastParams& P, Emit2 emit2) {
  constexpr int TS = Geo<HF>::TS;
  const int lgP = lgFT - 1, total = P.nb << lgP;
  for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
    const int kk = idx >> lgP, t0 = 2 * (idx & ((1 << lgP) - 1));
    if (t0 >= nf) continue;
    const float2 X0 = rfft_bin_fast<HF>(smem + t0 * TS, P.tw, P.klo + kk);
    const float2 X1 = t0 + 1 < nf ? rfft_bin_fast<HF>(smem + (t0 + 1) * TS, P.tw, P.klo + kk) : make_float2(0.f, 0.f);
    emit2(kk, t0, X0, X1, t0 + 1 < nf);
  }
}

// operand store of two adjacent focal points f, f + 1 (f even, ldf even): see store_operand
__device__ __forceinline__ void store_operand2(const OperandOut& O, int ld, int kk, int r, int f, float2 X0, float2 X1) {
  const int s = operand_row(O, r);
  if (s < 0) return;
  const size_t idx = ((size_t)kk * ld + s) * O.ldf + f;
  const float4 v = make_float4(X0.x, X0.y, X1.x, X1.y);
  *reinterpret_cast<float4*>(O.plain + idx) = v;
#pragma unroll
  for (int p = 0; p < kMaxPeers; ++p)
    if (p < O.npeer) *reinterpret_cast<float4*>(O.peer[p] + idx) = v;
}

// ------------------------------------------------------------------------------------------------ k_load_R_fast
// grid (ceil(nshots / ST), nrec); Rt: [nshots][nrec][nt]                                        (a0)
template <int HF>
__global__ void __launch_bounds__(256 * HF, 3 - HF)
k_load_R_fast(const float* __restrict__ Rt, float2* __restrict__ Rhat, FastParams P, int shot0, int nshots, int lgST) {
  extern __shared__ float2 smem[];
  pdl_trigger();  // the next kernel's CTAs may take the SMs this kernel's last wave leaves free ...
  warm_tables(P, P.warm != 0);
  pdl_wait();     // ... and this one touches global memory only after the kernel in front of it has completed
  constexpr int TS = Geo<HF>::TS;
  const int ST = 1 << lgST, r = P.r0 + blockIdx.y, g0 = blockIdx.x * ST;
  const int ns = min(ST, nshots - g0);
  const Who me = who<HF>();
  if (me.tl < ns) {
    float2 a[32];
    load_time<HF>(a, Rt + ((size_t)(g0 + me.tl) * P.n + r) * P.nt, me);
    float2* zt = smem + me.tl * TS;
    warp_fft1024<false>(a, zt + me.hf * SUB, P.tw1k, me.t);
    store_Z<HF>(a, zt, me.hf, me.t, P.tw);
  }
  __syncthreads();
  auto weight = [&](int s) { return __ldg(P.wscale + s); };
  if (lgST >= 2 && ((shot0 + g0) & 1) == 0) {
    band_out_pairs<HF>(smem, ns, lgST, P, [&](int kk, int t0, float2 X0, float2 X1, bool two) {
      const int s = shot0 + g0 + t0;  // even
      const float c0 = weight(s), c1 = two ? weight(s + 1) : 0.f;
      float2* dst = Rhat + rhat_index(P.tiled, r - P.r0, kk, s, P.nb, P.ld);  // s even: (s, s + 1) share one 16-byte chunk in either layout
      if (two) *reinterpret_cast<float4*>(dst) = make_float4(c0 * X0.x, c0 * X0.y, c1 * X1.x, c1 * X1.y);
      else *dst = make_float2(c0 * X0.x, c0 * X0.y);  // column s + 1 belongs to another chunk (or is padding)
    });
  } else {
    band_out<HF>(smem, ns, lgST, P, [&](int tl, int kk, float2 X) {
      const int s = shot0 + g0 + tl;
      const float sc = weight(s);
      Rhat[rhat_index(P.tiled, r - P.r0, kk, s, P.nb, P.ld)] = make_float2(sc * X.x, sc * X.y);
    });
  }
}

// ------------------------------------------------------------------------------------------------ k_fwd_fast
// grid (ceil(nfoc / FT), n); src: [nfoc][n][nt]                                                        (a1, a6)
template <int HF>
__global__ void __launch_bounds__(256 * HF, 3 - HF)
k_fwd_fast(const float* __restrict__ src, const __grid_constant__ OperandOut O, FastParams P, int lgFT, int conj_out, float* __restrict__ init_Tsrc) {
  extern __shared__ float2 smem[];
  pdl_trigger();  // the next kernel's CTAs may take the SMs this kernel's last wave leaves free ...
  warm_tables(P, P.warm != 0);
  pdl_wait();     // ... and this one touches global memory only after the kernel in front of it has completed
  constexpr int TS = Geo<HF>::TS;
  const int FT = 1 << lgFT, r = P.r0 + blockIdx.y, f0 = blockIdx.x * FT;
  const int nf = min(FT, P.nfoc - f0), nt = P.nt;
  const Who me = who<HF>();
  if (me.tl < nf) {
    float2 a[32];
    const size_t base = ((size_t)(f0 + me.tl) * P.n + r) * nt;
    load_time<HF>(a, src + base, me);
    if (init_Tsrc) {  // f1plus = N_{-1} = T G_d   [PAPER.md:19, 67, 74]
      float* dst = init_Tsrc + base;
#pragma unroll
      for (int q = 0; q < 32; ++q) {
        const int j = sample_j<HF>(q, me.t, me.hf);
        dst[(nt - j) & (nt - 1)] = a[q].x;
        dst[nt - j - 1] = a[q].y;
      }
    }
    float2* zt = smem + me.tl * TS;
    warp_fft1024<false>(a, zt + me.hf * SUB, P.tw1k, me.t);
    store_Z<HF>(a, zt, me.hf, me.t, P.tw);
  }
  __syncthreads();
  const float cs = conj_out ? -1.f : 1.f;  // conj: spectrum of the time-reversed real trace
  if (lgFT >= 2 && (O.ldf & 1) == 0) {
    band_out_pairs<HF>(smem, nf, lgFT, P, [&](int kk, int t0, float2 X0, float2 X1, bool) {
      store_operand2(O, P.ld, kk, r, f0 + t0, make_float2(X0.x, cs * X0.y), make_float2(X1.x, cs * X1.y));
    });
  } else {
    band_out<HF>(smem, nf, lgFT, P, [&](int tl, int kk, float2 X) { store_operand(O, P.ld, kk, r, f0 + tl, make_float2(X.x, cs * X.y)); });
  }
}

// ------------------------------------------------------------------------------------------------ k_inv_fast
// grid (ceil(nfoc / FT), n); spec: [n][nb][ldf]; out[j] = sS*S[j] + sA*A[j] + sB*B[(nt-j)%nt]              (a3, a7)
template <int HF>
__global__ void __launch_bounds__(256 * HF, 3 - HF)
k_inv_fast(const float2* __restrict__ spec, FastParams P, int lgFT, float* __restrict__ out, float sS,
           const float* __restrict__ A, float sA, const float* __restrict__ B, float sB) {
  extern __shared__ float2 smem[];
  pdl_trigger();  // the next kernel's CTAs may take the SMs this kernel's last wave leaves free ...
  warm_tables(P, P.warm != 0);
  pdl_wait();     // ... and this one touches global memory only after the kernel in front of it has completed
  constexpr int TS = Geo<HF>::TS;
  const int FT = 1 << lgFT, r = P.r0 + blockIdx.y, f0 = blockIdx.x * FT;
  const int nf = min(FT, P.nfoc - f0), nt = P.nt;
  const float2* srow = spec + (size_t)r * P.nb * P.ldf + f0;
  if (lgFT >= 2 && (P.ldf & 1) == 0 && simple_band(P, Geo<HF>::M)) {
    spectrum_in_pairs<HF, false>(smem, nf, lgFT, false, P, srow, nullptr);
  } else if (simple_band(P, Geo<HF>::M)) {
    spectrum_in_singles<HF, false>(smem, nf, lgFT, false, P, srow, nullptr);
  } else {
    spectrum_in<HF>(
        smem, nf, lgFT, false, P, [&](int tl, int kk, float2&) { return __ldg(srow + (size_t)kk * P.ldf + tl); },
        [](int, int, float2, float2) {});
  }
  __syncthreads();
  const Who me = who<HF>();
  if (me.tl >= nf) return;
  float2* zt = smem + me.tl * TS;
  float2 a[32];
  load_Z<HF>(a, zt, me.hf, me.t, P.tw);
  trace_sync<HF>(me.tl);
  warp_fft1024<true>(a, zt + me.hf * SUB, P.tw1k, me.t);
  const size_t base = ((size_t)(f0 + me.tl) * P.n + r) * nt;
#pragma unroll
  for (int q = 0; q < 32; ++q) {
    const int j = sample_j<HF>(q, me.t, me.hf);
    float2 v = make_float2(sS * a[q].x, sS * a[q].y);
    if (A) {
      const float2 av = __ldg(reinterpret_cast<const float2*>(A + base + j));
      v.x += sA * av.x;
      v.y += sA * av.y;
    }
    if (B) {
      v.x += sB * __ldg(B + base + ((nt - j) & (nt - 1)));
      v.y += sB * __ldg(B + base + (nt - j - 1));
    }
    *reinterpret_cast<float2*>(out + base + j) = v;
  }
}

// ------------------------------------------------------------------------------------------------ k_post_fast
// grid (ceil(nfoc / FT), n).  Shat, phat: [n][nb][ldf]; operand out: see store_operand; h: [nfoc][n];
// f1plus / f1min: [nfoc][n][nt].  One Neumann step after the contraction (a3..a6):
//   i even:  v = S (plain inverse transform);   w = Theta v;  f1min += w;   N_i = -T w  =>  N^_i = -conj(FFT w)
//   i odd:   u = T S (inverse of conj S^);      w = Theta u;  f1plus -= w;  N_i = -w    =>  N^_i = -FFT w
// (Theta is symmetric in +-t, so Theta T = T Theta; w is real, so FFT(T w) = conj FFT(w).)  Every global access of
// the time fields is a natural-order float2 row; only the optional N_i copy of an even step is written reversed.
template <int HF>
__global__ void __launch_bounds__(256 * HF, 3 - HF)
k_post_fast(const float2* __restrict__ Shat, float2* __restrict__ phat, const __grid_constant__ OperandOut O, const int* __restrict__ h,
            float* __restrict__ f1plus, float* __restrict__ f1min, FastParams P, int lgFT, int parity_even,
            float* __restrict__ Ni_out, int pf_dist) {
  extern __shared__ float2 smem[];
  pdl_trigger();  // the next kernel's CTAs may take the SMs this kernel's last wave leaves free ...
  warm_tables(P, P.warm != 0);
  pdl_wait();     // ... and this one touches global memory only after the kernel in front of it has completed
  constexpr int TS = Geo<HF>::TS;
  const int FT = 1 << lgFT, r = P.r0 + blockIdx.y, f0 = blockIdx.x * FT;
  const int nf = min(FT, P.nfoc - f0), nt = P.nt;
  const size_t rowoff = (size_t)r * P.nb * P.ldf + f0;
  const Who me = who<HF>();
  const bool pairs = lgFT >= 2 && (P.ldf & 1) == 0;
  if (pf_dist > 0) {
    // The S^ rows of the tile that takes this CTA's place on the SM (pf_dist = CTAs resident at once) start their way
    // from HBM to L2 now: its P1 then pays an L2 hit per round trip instead of a DRAM access behind everyone else's
    const long long L = (long long)blockIdx.y * gridDim.x + blockIdx.x + pf_dist;
    const int by = (int)(L / gridDim.x), bx = (int)(L - (long long)by * gridDim.x);
    if (by < (int)gridDim.y) {
      const size_t o = (size_t)(P.r0 + by) * P.nb * P.ldf + (size_t)bx * FT;
      for (int kk = threadIdx.x; kk < P.nb; kk += blockDim.x) asm volatile("prefetch.global.L2 [%0];" ::"l"(Shat + o + (size_t)kk * P.ldf));
    }
  }
  const int hh = me.tl < nf ? __ldg(h + (size_t)(f0 + me.tl) * P.n + r) : 0;
  // a3: p^ += S^   [PAPER.md:79]
  if (pairs && simple_band(P, Geo<HF>::M)) {
    spectrum_in_pairs<HF, true>(smem, nf, lgFT, parity_even == 0, P, Shat + rowoff, phat + rowoff);
  } else if (simple_band(P, Geo<HF>::M)) {
    spectrum_in_singles<HF, true>(smem, nf, lgFT, parity_even == 0, P, Shat + rowoff, phat + rowoff);
  } else {
    spectrum_in<HF>(
        smem, nf, lgFT, parity_even == 0, P,
        [&](int tl, int kk, float2& pv) {
          const size_t o = rowoff + (size_t)kk * P.ldf + tl;
          pv = phat[o];
          return __ldg(Shat + o);
        },
        [&](int tl, int kk, float2 s, float2 pv) { phat[rowoff + (size_t)kk * P.ldf + tl] = make_float2(pv.x + s.x, pv.y + s.y); });
  }
  __syncthreads();
  if (me.tl < nf) {
    float2* zt = smem + me.tl * TS;
    float2 a[32];
    load_Z<HF>(a, zt, me.hf, me.t, P.tw);
    trace_sync<HF>(me.tl);
    warp_fft1024<true>(a, zt + me.hf * SUB, P.tw1k, me.t);
    const size_t base = ((size_t)(f0 + me.tl) * P.n + r) * nt;
    float* acc = (parity_even ? f1min : f1plus) + base;
    const float sg = parity_even ? 1.f : -1.f;
    // a4 + a5.  Theta[j] = 1 iff j < h or j > nt - h (hard 0/1 window, strict inequality; G2).  Sample pairs that miss the
    // window touch no memory; the others are added to the accumulator by the L2 (red_add2: nothing is loaded).
#pragma unroll
    for (int q = 0; q < 32; ++q) {
      // register row q of the warp covers the samples [jlo, jhi]: a row that misses the window is cleared without a look
      const int jlo = sample_j<HF>(q, 0, me.hf), jhi = sample_j<HF>(q, 31, me.hf) + 1;
      if (jlo < hh || jhi > nt - hh) {  // warp-uniform
        const int j = sample_j<HF>(q, me.t, me.hf);
        const bool in0 = j < hh || j > nt - hh, in1 = j + 1 < hh || j + 1 > nt - hh;
        const float wx = in0 ? a[q].x : 0.f, wy = in1 ? a[q].y : 0.f;
        a[q] = make_float2(wx, wy);
        if (in0 || in1) red_add2(acc + j, sg * wx, sg * wy);
      } else {
        a[q] = make_float2(0.f, 0.f);
      }
    }
    if (Ni_out) {  // test / N_last copy of the new iterate
      float* ni = Ni_out + base;
#pragma unroll
      for (int q = 0; q < 32; ++q) {
        const int j = sample_j<HF>(q, me.t, me.hf);
        if (parity_even) {  // N_i[j'] = -w[(nt - j') % nt]
          ni[(nt - j) & (nt - 1)] = -a[q].x;
          ni[nt - j - 1] = -a[q].y;
        } else {
          *reinterpret_cast<float2*>(ni + j) = make_float2(-a[q].x, -a[q].y);
        }
      }
    }
    warp_fft1024<false>(a, zt + me.hf * SUB, P.tw1k, me.t);  // a6
    store_Z<HF>(a, zt, me.hf, me.t, P.tw);
  }
  __syncthreads();
  const float cs = parity_even ? 1.f : -1.f;
  if (pairs) {
    band_out_pairs<HF>(smem, nf, lgFT, P, [&](int kk, int t0, float2 X0, float2 X1, bool) {
      store_operand2(O, P.ld, kk, r, f0 + t0, make_float2(-X0.x, cs * X0.y), make_float2(-X1.x, cs * X1.y));
    });
  } else {
    band_out<HF>(smem, nf, lgFT, P, [&](int tl, int kk, float2 X) { store_operand(O, P.ld, kk, r, f0 + tl, make_float2(-X.x, cs * X.y)); });
  }
}

// ------------------------------------------------------------------------------------------------ host side
FastParams make_fast(const mk_ctx* c, int nfoc, int ldf) {
  FastParams P;
  P.tw = c->d_tw;
  P.tw1k = c->d_tw1k;
  P.wscale = c->d_wscale;
  P.nt = c->nt;
  P.n = c->n;
  P.nb = c->nb;
  P.klo = c->klo;
  P.ld = c->ld;
  P.ldf = ldf;
  P.nfoc = nfoc;
  P.tiled = c->rhat_layout;
  P.r0 = c->r0;
  P.warm = (c->tune & 8192) ? 0 : 1;
  return P;
}

struct Shape {
  int lg, threads;
  size_t smem;
};
// FT <= 8 traces per CTA (no more slots than traces), 32 HF threads per trace, at least 64 threads: with a single focal
// point the 2-warp CTAs of all receivers are resident at once (8 per SM at 128 registers) and the second warp shares
// the CTA-wide phases P1 / P5.  Measured on config 1 (601 traces per launch): 256 threads 29 us (3 waves), 32 threads 40 us
Shape shape_for(const mk_ctx* c, int count) {
  const int HF = c->nt / 2048;
  int lg = HF == 1 || (c->tune & 2048) ? 3 : 2;  // 256 threads and <= 68 KB of traces per CTA: two CTAs per SM overlap each other's memory phases
                                                 // (MK_OPT_TUNE bit 11: nt = 4096 with eight traces = 512 threads, one CTA per SM)
  while (lg > 0 && (1 << (lg - 1)) >= count) --lg;
  Shape s;
  s.lg = lg;
  s.threads = std::max(32 * HF << lg, 64);
  s.smem = ((size_t)(HF * SUB + 2) << lg) * sizeof(float2);
  return s;
}

template <typename K>
int set_smem(mk_ctx* c, K kernel, size_t bytes) {
  return check_cuda(c, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes), "cudaFuncSetAttribute");
}

}  // namespace

bool fast_fft_ok(const mk_ctx* c) { return (c->nt == 2048 || c->nt == 4096) && c->fft_path != 1 && c->d_tw1k != nullptr; }

#define MK_FAST_LAUNCH(KERN, GRID, SH, ...)                                          \
  do {                                                                               \
    if (c->nt == 2048) {                                                             \
      if (int rc = set_smem(c, KERN<1>, (SH).smem)) return rc;                       \
      if (int rc = check_cuda(c, launch_pdl(c, KERN<1>, GRID, (SH).threads, (SH).smem, __VA_ARGS__), #KERN)) return rc; \
    } else {                                                                         \
      if (int rc = set_smem(c, KERN<2>, (SH).smem)) return rc;                       \
      if (int rc = check_cuda(c, launch_pdl(c, KERN<2>, GRID, (SH).threads, (SH).smem, __VA_ARGS__), #KERN)) return rc; \
    }                                                                                \
    ++c->launches;                                                                   \
    return check_cuda(c, cudaGetLastError(), #KERN);                                 \
  } while (0)

int launch_load_R_fast(mk_ctx* c, const RowBlock& rb, const float* d_R_time, int shot0, int nshots) {
  const Shape sh = shape_for(c, nshots);
  const dim3 grid((nshots + (1 << sh.lg) - 1) >> sh.lg, rb.nrow);
  FastParams P = make_fast(c, 0, 0);
  P.r0 = rb.r0;
  if (rb.ld) P.ld = rb.ld;
  if (rb.src_n) P.n = rb.src_n;
  MK_FAST_LAUNCH(k_load_R_fast, grid, sh, d_R_time, rb.Rhat, P, shot0, nshots, sh.lg);
}

int launch_fwd_fast(mk_ctx* c, const float* d_src, const OperandOut& O, int nfoc, bool conj_out, float* d_init_Tsrc) {
  const Shape sh = shape_for(c, nfoc);
  const dim3 grid((nfoc + (1 << sh.lg) - 1) >> sh.lg, c->nrow);
  MK_FAST_LAUNCH(k_fwd_fast, grid, sh, d_src, O, make_fast(c, nfoc, O.ldf), sh.lg, conj_out ? 1 : 0, d_init_Tsrc);
}

int launch_inv_fast(mk_ctx* c, const float2* d_spec, int nfoc, int ldf, float* d_out, float sS, const float* d_A, float sA,
                    const float* d_B, float sB) {
  const Shape sh = shape_for(c, nfoc);
  const dim3 grid((nfoc + (1 << sh.lg) - 1) >> sh.lg, c->nrow);
  MK_FAST_LAUNCH(k_inv_fast, grid, sh, d_spec, make_fast(c, nfoc, ldf), sh.lg, d_out, sS, d_A, sA, d_B, sB);
}

int launch_post_fast(mk_ctx* c, const OperandOut& O, int parity_even, float* d_Ni_out) {
  const Shape sh = shape_for(c, c->nfoc);
  const dim3 grid((c->nfoc + (1 << sh.lg) - 1) >> sh.lg, c->nrow);
  // CTAs resident at once (registers: 128 per thread; shared memory): the distance of the L2 prefetch of the next tile's spectra
  const int per_sm = std::max<int>(1, std::min<size_t>(std::min<size_t>(65536 / (128 * sh.threads), (c->smem_sm ? c->smem_sm : 233472) / (sh.smem + 1024)), 32));
  const long long total = (long long)grid.x * grid.y;
  const int pf_dist = !(c->tune & 1) && total > (long long)per_sm * c->num_sms ? per_sm * c->num_sms : 0;
  MK_FAST_LAUNCH(k_post_fast, grid, sh, c->d_Shat, c->d_phat, O, c->d_h, c->acc_plus, c->acc_min, make_fast(c, c->nfoc, c->ldf),
                 sh.lg, parity_even, d_Ni_out, pf_dist);
}

}  // namespace mk

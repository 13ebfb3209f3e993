// mk_api.cu — the C ABI of include/mk.h: argument checks, device buffers, and the order of kernel launches.
// No arithmetic of the method happens on the host: every step of SURVEY.md §8(a) is a kernel in
// mk_fft_kernels.cu / mk_syn_gemv.cu / mk_syn_gemm.cu.  There is no CPU fallback.
#include <cuda.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>

#include "mk_fft_common.cuh"

namespace mk {

int set_err(mk_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg;
  return code;
}

int check_cuda(mk_ctx* c, cudaError_t e, const char* what) {
  if (e == cudaSuccess) return MK_OK;
  if (c) {
    c->sticky = MK_ERR_CUDA;
    c->err = std::string(what) + ": " + cudaGetErrorString(e);
  }
  return e == cudaErrorMemoryAllocation ? MK_ERR_OOM : MK_ERR_CUDA;
}

namespace {

template <typename T>
int ensure(mk_ctx* c, T** p, size_t* cap, size_t count, const char* what) {
  if (*cap >= count && *p) return MK_OK;
  if (*p) {
    cudaFree(*p);
    c->device_bytes -= *cap * sizeof(T);
    *p = nullptr;
    *cap = 0;
  }
  void* q = nullptr;
  cudaError_t e = cudaMalloc(&q, count * sizeof(T));
  if (e != cudaSuccess) {
    cudaGetLastError();
    char buf[160];
    snprintf(buf, sizeof buf, "cudaMalloc(%s, %zu bytes) failed: %s", what, count * sizeof(T), cudaGetErrorString(e));
    return set_err(c, MK_ERR_OOM, buf);
  }
  *p = static_cast<T*>(q);
  *cap = count;
  c->device_bytes += count * sizeof(T);
  return MK_OK;
}

template <typename T>
void release(mk_ctx* c, T** p, size_t* cap) {
  if (*p) {
    cudaFree(*p);
    c->device_bytes -= *cap * sizeof(T);
  }
  *p = nullptr;
  *cap = 0;
}

int resolve_regime(mk_ctx* c, int nfoc, int* regime) {
  int r = c->regime;
  if (c->rhat_format == 1) {  // compressed R^ serves the bandwidth-bound regime only
    if (!gemv_supported(c, nfoc) || r > 1) return set_err(c, MK_ERR_INVALID_ARG, "compressed R^ (MK_OPT_RHAT_FORMAT = 1) needs the streaming regime: nfoc <= 8");
    r = 1;
  }
  if (c->rhat_layout == 1) {  // tiled R^ is read by the tcgen05 contraction only
    if (r != 0 && r != 3) return set_err(c, MK_ERR_INVALID_ARG, "tiled R^ (MK_OPT_RHAT_LAYOUT = 1) is read by the tcgen05 regime only");
    r = 3;
  }
  if (r == 0) r = gemv_supported(c, nfoc) ? 1 : (tc_supported(c) ? 3 : 2);
  if (r == 1 && !gemv_supported(c, nfoc)) return set_err(c, MK_ERR_INVALID_ARG, "GEMV regime needs nfoc <= 8 and ld*nfoc*8 <= 96 KiB");
  if (r < 1 || r > 3) return set_err(c, MK_ERR_INVALID_ARG, "unknown regime");
  if (r == 3 && !tc_supported(c)) return set_err(c, MK_ERR_INVALID_ARG, "tcgen05 3xTF32 regime needs an sm_100 device");
  *regime = r;
  return MK_OK;
}

// columns of N^ / S^ / p^ per bin row: the GEMV reads nfoc, the FFMA GEMM 128-bit pairs, the tcgen05 GEMM 32-float TMA boxes
inline int ldf_for(int regime, int nfoc) { return regime == 1 ? nfoc : (regime == 2 ? ((nfoc + 3) / 4) * 4 : ((nfoc + 15) / 16) * 16); }

// the operand of slot 0 (the run) or 1 (scratch: mk_synthesis, finals)
OperandOut operand_out(mk_ctx* c, int slot, int ldf) {
  OperandOut O{};
  O.ldf = ldf;
  O.plain = slot ? c->d_Nhat2 : c->d_Nhat;
  O.shot_of_rec = c->d_shot_of_rec;
  if (c->npeer[slot] > 0 && c->peer_key[slot] == c->operand_key[slot] && c->operand_key[slot] != 0) {
    O.npeer = c->npeer[slot];
    for (int p = 0; p < O.npeer; ++p) O.peer[p] = reinterpret_cast<float2*>(c->peer_plane[slot][p]);
  }
  return O;
}

// allocate the operand of a slot; zero it when the buffer is new or its layout changed.  Pad rows / columns must be
// zero and no kernel ever writes a non-zero there (the forward transforms store rows r < n, columns f < nfoc, and zeros
// into the odd pad column of a pair), so an operand that keeps its layout needs no second memset.
int prepare_operand(mk_ctx* c, int slot, int nfoc, int ldf) {
  const long long key = ((long long)nfoc << 32) ^ (long long)ldf;
  const size_t nN = (size_t)c->nb * c->ld * ldf;
  float2** p = slot ? &c->d_Nhat2 : &c->d_Nhat;
  size_t* cap = slot ? &c->cap_Nhat2 : &c->cap_Nhat;
  const float2* before = *p;
  if (int rc = ensure(c, p, cap, nN, "Nhat")) return rc;
  if (*p == before && c->operand_key[slot] == key) return MK_OK;
  c->operand_key[slot] = 0;
  if (int rc = check_cuda(c, cudaMemsetAsync(*p, 0, nN * sizeof(float2), c->stream), "memset Nhat")) return rc;
  c->operand_key[slot] = key;
  return MK_OK;
}

// Out-of-core R^ (mk_create_streamed; "synthesis must be done in a batched fashion ... a certain batch is
// transferred to each GPU", Algorithm 2's copyH2D_shot_batch loop PAPER.md:98-112, the 249 GB case PAPER.md:42): the rows
// of R^ that do not fit are kept in pinned host memory and every contraction pulls them through two windows in HBM, one
// cudaMemcpyAsync per row block on a copy stream, the contraction of block b overlapping the transfer of block b + 1.
// Row blocks are independent (every output trace depends on one row of R^), so the result is that of the
// resident contraction bit for bit.  Consecutive passes walk the blocks in opposite directions: the two blocks left in
// the windows by one pass are the first two of the next and are not transferred again.
template <typename Launch>
int stream_host_rows(mk_ctx* c, Launch&& launch, const RowBlock& resident) {
  const int nhost = c->nrow - c->nres, W = c->win_rows, B = (nhost + W - 1) / W;
  // the copy stream starts behind everything enqueued so far (ingest into the host rows, earlier uses of the windows)
  if (int rc = check_cuda(c, cudaEventRecord(c->win_main, c->stream), "cudaEventRecord")) return rc;
  if (int rc = check_cuda(c, cudaStreamWaitEvent(c->h2d_stream, c->win_main, 0), "cudaStreamWaitEvent")) return rc;
  const size_t row_elems = (size_t)c->nb * c->ld;
  auto fetch = [&](int b) -> int {  // enqueue the transfer of block b unless its window already holds it
    const int buf = b & 1;
    if (c->win_block[buf] == b) return MK_OK;
    const int rows = std::min(W, nhost - b * W);
    if (c->win_block[buf] >= 0)  // the contraction that last read this window (this pass or an earlier one)
      if (int rc = check_cuda(c, cudaStreamWaitEvent(c->h2d_stream, c->win_free[buf], 0), "cudaStreamWaitEvent")) return rc;
    c->win_block[buf] = -1;
    const size_t bytes = (size_t)rows * row_elems * sizeof(float2);
    if (int rc = check_cuda(c, cudaMemcpyAsync(c->d_win[buf], c->h_Rhat + (size_t)b * W * row_elems, bytes, cudaMemcpyHostToDevice, c->h2d_stream),
                            "H2D row block of R^"))
      return rc;
    if (int rc = check_cuda(c, cudaEventRecord(c->win_ready[buf], c->h2d_stream), "cudaEventRecord")) return rc;
    c->win_block[buf] = b;
    c->h2d_bytes += (double)bytes;
    return MK_OK;
  };
  auto block_at = [&](int i) { return c->win_reverse ? B - 1 - i : i; };
  if (int rc = fetch(block_at(0))) return rc;
  if (B > 1)
    if (int rc = fetch(block_at(1))) return rc;
  if (resident.nrow > 0)  // runs while the first blocks arrive
    if (int rc = launch(resident)) return rc;
  for (int i = 0; i < B; ++i) {
    const int b = block_at(i), buf = b & 1, rows = std::min(W, nhost - b * W);
    if (int rc = check_cuda(c, cudaStreamWaitEvent(c->stream, c->win_ready[buf], 0), "cudaStreamWaitEvent")) return rc;
    if (int rc = launch(RowBlock{c->d_win[buf], c->nres + b * W, rows})) return rc;
    if (int rc = check_cuda(c, cudaEventRecord(c->win_free[buf], c->stream), "cudaEventRecord")) return rc;
    if (i + 2 < B)
      if (int rc = fetch(block_at(i + 2))) return rc;
  }
  c->win_reverse = !c->win_reverse;
  return MK_OK;
}

// a2: S^ = R^ x N^ per bin, on the context's stream; optionally bracketed by events
// peers attached for another operand layout would silently receive nothing: refuse to produce rows then
int check_peers(mk_ctx* c, int slot) {
  if (c->npeer[slot] > 0 && c->peer_key[slot] != c->operand_key[slot])
    return set_err(c, MK_ERR_STATE, "the operand layout changed since mk_operand_attach: reserve and attach again");
  return MK_OK;
}

int contract(mk_ctx* c, int slot, float2* Shat, int nfoc, int ldf, int regime) {
  if (c->operand_stale[slot])
    return set_err(c, MK_ERR_STATE, "row-sharded context: the operand rows were not exchanged (mk_operand / mk_operand_exchanged)");
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  bool timed = c->timing > 0 && c->syn_count % (size_t)c->timing == 0;   // MK_OPT_TIMING = N: every N-th contraction
  ++c->syn_count;
  if (timed && c->ev_used + 2 > c->ev.size()) {
    if (c->ev.size() >= 65536) timed = false;  // pool full: later launches go untimed (read / reset the counters)
    else
      for (int i = 0; i < 2; ++i) {
        cudaEvent_t e;
        if (int rc = check_cuda(c, cudaEventCreate(&e), "cudaEventCreate")) return rc;
        c->ev.push_back(e);
      }
  }
  if (timed) {
    e0 = c->ev[c->ev_used];
    e1 = c->ev[c->ev_used + 1];
    c->ev_used += 2;
    cudaEventRecord(e0, c->stream);
  }
  const float2* Nhat = slot ? c->d_Nhat2 : c->d_Nhat;
  auto launch = [&](const RowBlock& rb) -> int {
    if (c->rhat_format == 1) return launch_syn_gemv_q16(c, Nhat, Shat, nfoc);
    if (regime == 1) return launch_syn_gemv(c, rb, Nhat, Shat, nfoc);
    if (regime == 2) return launch_syn_gemm(c, rb, Nhat, Shat, ldf);
    return launch_syn_tc(c, rb, slot, Nhat, Shat, ldf);
  };
  int rc = MK_OK;
  if (c->nres < c->nrow) rc = stream_host_rows(c, launch, /*before the first block arrives:*/ RowBlock{c->d_Rhat, c->r0, c->nres});
  else rc = launch(RowBlock{c->d_Rhat, c->r0, c->nrow});
  if (timed) cudaEventRecord(e1, c->stream);
  c->last_regime = regime;  // information only (MK_INFO_REGIME_USED); the run's regime is c->run_regime
  return rc;
}

bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }

// Calls that change what a run was started from (R^, eps, the operand layout) END the run in progress: the next
// mk_step / mk_finish returns MK_ERR_STATE until mk_begin.  Between the two halves of a step they are refused.
int end_run(mk_ctx* c, const char* who) {
  if (c->contracted) return set_err(c, MK_ERR_STATE, std::string(who) + " between mk_step_contract and mk_step_post");
  c->begun = false;
  c->prepared_field = 0;
  return MK_OK;
}

bool overlaps(const void* a, const void* b, size_t bytes) {
  if (!a || !b) return false;
  const char* x = static_cast<const char*>(a);
  const char* y = static_cast<const char*>(b);
  return x < y + bytes && y < x + bytes;
}

// quadrature weights of the shot grid (folded into R^ at ingest as dt * w[s]) and the receiver -> shot map of the
// operand rows.  h_w == nullptr: trapezoid rule with spacing dx over the ns shots; h_rec_of_shot == nullptr: shot s is
// co-located with receiver s (for s < min(ns, n); further shots have no receiver, further receivers no shot).
int upload_geometry(mk_ctx* c, const int* h_rec_of_shot, const float* h_w) {
  std::vector<float> ws(c->ns);
  for (int s = 0; s < c->ns; ++s) {
    const double w = h_w ? (double)h_w[s] : ((c->ns > 1 && (s == 0 || s == c->ns - 1)) ? 0.5 * c->dx : c->dx);
    if (!(w >= 0.0) || !std::isfinite(w)) return set_err(c, MK_ERR_INVALID_ARG, "mk_set_geometry: weights must be finite and >= 0");
    ws[s] = (float)(c->dt * w);
  }
  std::vector<int> sor(c->n, -1);
  bool identity = c->ns == c->n;
  for (int s = 0; s < c->ns; ++s) {
    const int r = h_rec_of_shot ? h_rec_of_shot[s] : (s < c->n ? s : -1);
    if (r < -1 || r >= c->n) return set_err(c, MK_ERR_INVALID_ARG, "mk_set_geometry: rec_of_shot out of range");
    if (r >= 0) {
      if (sor[r] != -1) return set_err(c, MK_ERR_INVALID_ARG, "mk_set_geometry: two shots at one receiver");
      sor[r] = s;
    }
    identity = identity && r == s;
  }
  if (!c->d_wscale) {
    size_t cap = 0;
    if (int rc = ensure(c, &c->d_wscale, &cap, (size_t)c->ns, "weights")) return rc;
  }
  if (int rc = check_cuda(c, cudaMemcpy(c->d_wscale, ws.data(), ws.size() * sizeof(float), cudaMemcpyHostToDevice), "weights upload")) return rc;
  if (identity) {  // the kernels take the receiver index itself
    if (c->d_shot_of_rec) {
      cudaFree(c->d_shot_of_rec);
      c->device_bytes -= (size_t)c->n * sizeof(int);
      c->d_shot_of_rec = nullptr;
    }
    return MK_OK;
  }
  if (!c->d_shot_of_rec) {
    size_t cap = 0;
    if (int rc = ensure(c, &c->d_shot_of_rec, &cap, (size_t)c->n, "receiver -> shot map")) return rc;
  }
  return check_cuda(c, cudaMemcpy(c->d_shot_of_rec, sor.data(), sor.size() * sizeof(int), cudaMemcpyHostToDevice), "map upload");
}

// outputs of the finals (and N_last) are written while the accumulators are still being read: they must not overlap
// f1plus / f1min (the caller's fields when mk_run accumulates in them, else the library's)
int check_output_alias(mk_ctx* c, const mk_outputs* o, const float* acc_plus, const float* acc_min, size_t bytes) {
  const float* outs[4] = {o->N_last, o->G, o->Gplus, o->Gminus};
  for (const float* p : outs)
    if (overlaps(p, acc_plus, bytes) || overlaps(p, acc_min, bytes))
      return set_err(c, MK_ERR_INVALID_ARG, "N_last / G / Gplus / Gminus must not overlap the f1plus / f1min fields");
  return MK_OK;
}

// NEXT-1 imaging: image[f] = dt * sum_r w[r] sum_j G^-[f][r][(nt-j)%nt] f1plus[f][r][j], the zero-time sample of the
// convolution of G^- with f1plus summed over the receivers [PAPER.md:24, 89].  Neither field is band-limited (the window
// Theta is applied in time), so the sum is taken over the time samples; it is a plain dot product of two fields and
// HBM-bound: grid (focal point, receiver chunk), coalesced forward reads of f1plus and coalesced backward reads of G^-,
// 8 independent loads per thread in flight, fp32 per (thread, receiver), double across receivers, fixed-order two-stage
// reduction (bit-reproducible).
constexpr int kImgThreads = 256;

__global__ void __launch_bounds__(kImgThreads)
k_image_partial(const float* __restrict__ Gminus, const float* __restrict__ f1plus, double* __restrict__ part, int n, int nt,
                int rows_per_cta, float w_mid, float w_end) {
  const int f = blockIdx.x, r0 = blockIdx.y * rows_per_cta, r1 = min(n, r0 + rows_per_cta);
  const int tid = threadIdx.x, mask = nt - 1;
  double acc = 0.0;
  for (int r = r0; r < r1; ++r) {
    const float* g = Gminus + ((size_t)f * n + r) * nt;
    const float* p = f1plus + ((size_t)f * n + r) * nt;
    float s[4] = {0.f, 0.f, 0.f, 0.f};
    int j = tid;
    for (; j + 3 * kImgThreads < nt; j += 4 * kImgThreads) {
      float gv[4], pv[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        pv[u] = __ldg(p + j + u * kImgThreads);
        gv[u] = __ldg(g + ((nt - j - u * kImgThreads) & mask));
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) s[u] = fmaf(gv[u], pv[u], s[u]);
    }
    for (; j < nt; j += kImgThreads) s[0] = fmaf(__ldg(g + ((nt - j) & mask)), __ldg(p + j), s[0]);
    const float w = (n > 1 && (r == 0 || r == n - 1)) ? w_end : w_mid;
    acc += (double)(w * ((s[0] + s[1]) + (s[2] + s[3])));
  }
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
  __shared__ double red[kImgThreads / 32];
  if ((tid & 31) == 0) red[tid >> 5] = acc;
  __syncthreads();
  if (tid == 0) {
    double t = 0.0;
    for (int i = 0; i < kImgThreads / 32; ++i) t += red[i];
    part[(size_t)f * gridDim.y + blockIdx.y] = t;
  }
}

__global__ void k_image_final(const double* __restrict__ part, float* __restrict__ image, int nfoc, int nchunk) {
  const int f = blockIdx.x * blockDim.x + threadIdx.x;
  if (f >= nfoc) return;
  double t = 0.0;
  for (int i = 0; i < nchunk; ++i) t += part[(size_t)f * nchunk + i];
  image[f] = (float)t;
}

}  // namespace
}  // namespace mk

using namespace mk;

// every entry point: reject a null / poisoned context and make the context's device current (the caller may have
// switched devices between calls; kernels, allocations and IPC opens must go to the GPU the context lives on)
#define MK_GUARD(ctx)                                          \
  if (!(ctx)) return MK_ERR_INVALID_ARG;                       \
  if ((ctx)->sticky) return (ctx)->sticky;                     \
  if (cudaSetDevice((ctx)->dev) != cudaSuccess) {              \
    cudaGetLastError();                                        \
    return set_err((ctx), MK_ERR_CUDA, "cudaSetDevice failed"); \
  }

// ---- mk_image_static: scratch of the imaging kernels for callers that cannot allocate --------------------------------
// The per (focal point, receiver chunk) partial sums of k_image_partial in a file-scope array instead of a cudaMalloc'ed
// buffer: part of the module image, so every GPU that loads libmk.so holds these 128 KB until the process exits.  In host
// code the NAME of the array is only a host-side stand-in, never a device address: its address on each device is asked for
// once (cudaGetSymbolAddress with that device current) and kept per device.  All calls on a device share the array.
static __device__ __align__(256) double g_image_static_part[MK_IMAGE_STATIC_MAX_PARTIALS];

namespace {
constexpr int kMaxStaticDevices = 64;
std::mutex g_image_static_mu;
double* g_image_static_ptr[kMaxStaticDevices] = {};   // [device] -> device address of g_image_static_part, or null

// called with the context's device current (MK_GUARD); no allocation: the array exists since the module was loaded
int image_static_scratch(mk_ctx* c, double** out) {
  if (c->dev < 0 || c->dev >= kMaxStaticDevices) return set_err(c, MK_ERR_INVALID_ARG, "mk_image_static: device ordinal beyond 63");
  std::lock_guard<std::mutex> lk(g_image_static_mu);
  if (!g_image_static_ptr[c->dev]) {
    double* p = nullptr;
    if (int rc = check_cuda(c, cudaGetSymbolAddress((void**)&p, g_image_static_part), "cudaGetSymbolAddress(g_image_static_part)")) return rc;
    if (!p) return set_err(c, MK_ERR_CUDA, "cudaGetSymbolAddress returned a null address for g_image_static_part");
    g_image_static_ptr[c->dev] = p;
  }
  *out = g_image_static_ptr[c->dev];
  return MK_OK;
}
}  // namespace

extern "C" {

const char* mk_version(void) { return "libmk 0.1 (sm_100a)"; }

const char* mk_last_error(mk_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

static int create_impl(mk_ctx** out, int nshot, int nrec, int nt, double dt, double dx, double fmin, double fmax, int row0,
                       int nrows, int resident_rows, int window_rows);

int mk_create(mk_ctx** out, int nshot, int nrec, int nt, double dt, double dx, double fmin, double fmax) {
  return create_impl(out, nshot, nrec, nt, dt, dx, fmin, fmax, 0, nrec, nrec, 0);
}

int mk_create_sharded(mk_ctx** out, int nshot, int nrec, int nt, double dt, double dx, double fmin, double fmax, int row0,
                      int nrows) {
  return create_impl(out, nshot, nrec, nt, dt, dx, fmin, fmax, row0, nrows, nrows, 0);
}

int mk_create_streamed(mk_ctx** out, int nshot, int nrec, int nt, double dt, double dx, double fmin, double fmax,
                       int resident_rows, int window_rows) {
  if (!out) return MK_ERR_INVALID_ARG;
  *out = nullptr;
  if (resident_rows < 0 || resident_rows > nrec || window_rows < 0) return MK_ERR_INVALID_ARG;
  return create_impl(out, nshot, nrec, nt, dt, dx, fmin, fmax, 0, nrec, resident_rows, window_rows);
}

static int create_impl(mk_ctx** out, int nshot, int nrec, int nt, double dt, double dx, double fmin, double fmax, int row0,
                       int nrows, int resident_rows, int window_rows) {
  if (!out) return MK_ERR_INVALID_ARG;
  *out = nullptr;
  if (nshot <= 0 || nrec <= 0) return MK_ERR_INVALID_ARG;
  if (row0 < 0 || nrows <= 0 || row0 + nrows > nrec) return MK_ERR_INVALID_ARG;
  if (nrows != nrec && nshot != nrec) return MK_ERR_INVALID_ARG;  // row sharding exchanges operand rows by receiver index: co-located spreads only
  if (!is_pow2(nt) || nt < 16 || nt > 32768) return MK_ERR_INVALID_ARG;
  if (!(dt > 0.0) || !(dx > 0.0) || !(fmin >= 0.0) || !(fmax >= fmin) || fmax > 0.5 / dt * (1.0 + 1e-9)) return MK_ERR_INVALID_ARG;
  int dev = 0, ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return MK_ERR_CUDA;  // no CPU fallback
  }
  mk_ctx* c = new (std::nothrow) mk_ctx();
  if (!c) return MK_ERR_OOM;
  *out = c;  // returned even on failure so that mk_last_error can be read; the caller destroys it
  c->n = nrec;
  c->ns = nshot;
  c->r0 = row0;
  c->nrow = nrows;
  c->nt = nt;
  c->dt = dt;
  c->dx = dx;
  c->fmin = fmin;
  c->fmax = fmax;
  // band B (reading G8): inclusive edges with a 1e-6-bin guard against rounding of 1/(nt dt)
  const double df = 1.0 / ((double)nt * dt);
  int lo = (int)std::ceil(fmin / df - 1e-6), hi = (int)std::floor(fmax / df + 1e-6);
  if (lo < 0) lo = 0;
  if (hi > nt / 2) hi = nt / 2;
  if (hi < lo) return set_err(c, MK_ERR_INVALID_ARG, "empty band");
  c->klo = lo;
  c->khi = hi;
  c->nb = hi - lo + 1;
  c->ld = ((nshot + 15) / 16) * 16;
  c->plan = mkfft::make_plan(nt);
  if (int rc = check_cuda(c, cudaGetDevice(&dev), "cudaGetDevice")) return rc;
  c->dev = dev;
  int v = 0;
  cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev);
  c->num_sms = v;
  cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  c->smem_optin = (size_t)v;
  cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev);
  c->smem_sm = (size_t)v;
  c->shot_loaded.assign(nshot, 0);
  if (int rc = upload_geometry(c, nullptr, nullptr)) return rc;  // trapezoid weights; shot s at receiver s
  // twiddles e^{-2 pi i k / nt}, evaluated in double (table constants only)
  {
    std::vector<float2> tw(nt);
    const double two_pi = 6.283185307179586476925286766559;
    for (int k = 0; k < nt; ++k) {
      const double a = -two_pi * (double)k / (double)nt;
      tw[k] = make_float2((float)std::cos(a), (float)std::sin(a));
    }
    size_t cap = 0;
    if (int rc = ensure(c, &c->d_tw, &cap, (size_t)nt, "twiddles")) return rc;
    if (int rc = check_cuda(c, cudaMemcpy(c->d_tw, tw.data(), nt * sizeof(float2), cudaMemcpyHostToDevice), "twiddle upload")) return rc;
  }
  {  // middle twiddles of the register-resident path: W_1024^{k1 t}, table constants evaluated in double
    std::vector<float2> tw(1024);
    const double two_pi = 6.283185307179586476925286766559;
    for (int k1 = 0; k1 < 32; ++k1)
      for (int t = 0; t < 32; ++t) {
        const double a = -two_pi * (double)(k1 * t) / 1024.0;
        tw[k1 * 32 + t] = make_float2((float)std::cos(a), (float)std::sin(a));
      }
    size_t cap = 0;
    if (int rc = ensure(c, &c->d_tw1k, &cap, (size_t)1024, "twiddles 1k")) return rc;
    if (int rc = check_cuda(c, cudaMemcpy(c->d_tw1k, tw.data(), 1024 * sizeof(float2), cudaMemcpyHostToDevice), "twiddle upload")) return rc;
  }
  c->nres = resident_rows;
  if (c->nres > 0) {
    size_t cap = 0;
    c->rhat_rows_alloc = c->nres;
    const size_t cnt = (size_t)c->nres * c->nb * c->ld;  // the rows this context owns and keeps in HBM
    if (int rc = ensure(c, &c->d_Rhat, &cap, cnt, "Rhat")) return rc;
    if (int rc = check_cuda(c, cudaMemset(c->d_Rhat, 0, cnt * sizeof(float2)), "Rhat memset")) return rc;
  }
  if (c->nres < nrows) {  // out-of-core: the other rows in pinned, device-mapped host memory + two windows in HBM
    const int nhost = nrows - c->nres;
    c->win_rows = window_rows > 0 ? std::min(window_rows, nhost) : std::max(1, (nhost + 7) / 8);
    const size_t row_elems = (size_t)c->nb * c->ld, host_bytes = (size_t)nhost * row_elems * sizeof(float2);
    void* hp = nullptr;
    if (cudaHostAlloc(&hp, host_bytes, cudaHostAllocMapped) != cudaSuccess) {
      cudaGetLastError();
      return set_err(c, MK_ERR_OOM, "cudaHostAlloc of the host-resident rows of R^ failed");
    }
    c->h_Rhat = static_cast<float2*>(hp);
    std::memset(hp, 0, host_bytes);  // pad columns stay zero
    void* dp = nullptr;
    if (int rc = check_cuda(c, cudaHostGetDevicePointer(&dp, hp, 0), "cudaHostGetDevicePointer")) return rc;
    c->h_Rhat_dev = static_cast<float2*>(dp);
    const int nwin = nhost > c->win_rows ? 2 : 1;
    for (int i = 0; i < nwin; ++i) {
      size_t cap = 0;
      if (int rc = ensure(c, &c->d_win[i], &cap, (size_t)c->win_rows * row_elems, "R^ window")) return rc;
    }
    if (int rc = check_cuda(c, cudaStreamCreateWithFlags(&c->h2d_stream, cudaStreamNonBlocking), "cudaStreamCreate")) return rc;
    for (int i = 0; i < 2; ++i) {
      if (int rc = check_cuda(c, cudaEventCreateWithFlags(&c->win_ready[i], cudaEventDisableTiming), "cudaEventCreate")) return rc;
      if (int rc = check_cuda(c, cudaEventCreateWithFlags(&c->win_free[i], cudaEventDisableTiming), "cudaEventCreate")) return rc;
    }
    if (int rc = check_cuda(c, cudaEventCreateWithFlags(&c->win_main, cudaEventDisableTiming), "cudaEventCreate")) return rc;
  }
  return MK_OK;
}

int mk_destroy(mk_ctx* c) {
  if (!c) return MK_OK;
  cudaFree(c->d_tw);
  cudaFree(c->d_tw1k);
  cudaFree(c->d_Rhat);
  cudaFree(c->d_wscale);
  cudaFree(c->d_shot_of_rec);
  cudaFree(c->d_f1plus);
  cudaFree(c->d_f1min);
  cudaFree(c->d_Nhat);
  cudaFree(c->d_Shat);
  cudaFree(c->d_phat);
  cudaFree(c->d_h);
  cudaFree(c->d_Nhat2);
  cudaFree(c->d_Shat2);
  cudaFree(c->d_stage);
  cudaFree(c->d_Rq);
  cudaFree(c->d_Rscale);
  cudaFree(c->d_qstage);
  cudaFree(c->d_img_part);
  cudaFree(c->d_tc_progress);
  cudaFree(c->d_sync_flags);
  cudaFree(c->d_win[0]);
  cudaFree(c->d_win[1]);
  if (c->h2d_stream) {
    cudaStreamSynchronize(c->h2d_stream);
    cudaStreamDestroy(c->h2d_stream);
  }
  for (int i = 0; i < 2; ++i) {
    if (c->win_ready[i]) cudaEventDestroy(c->win_ready[i]);
    if (c->win_free[i]) cudaEventDestroy(c->win_free[i]);
  }
  if (c->win_main) cudaEventDestroy(c->win_main);
  if (c->h_Rhat) cudaFreeHost(c->h_Rhat);
  if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  if (c->copy_ev) cudaEventDestroy(c->copy_ev);
  for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
  cudaGetLastError();
  delete c;
  return MK_OK;
}

int mk_set_stream(mk_ctx* c, void* cuda_stream) {
  MK_GUARD(c);
  c->stream = static_cast<cudaStream_t>(cuda_stream);
  return MK_OK;
}

int mk_set_option(mk_ctx* c, int key, double value) {
  MK_GUARD(c);
  switch (key) {
    case MK_OPT_EPS_SAMPLES:
      if (value < 0 || value > c->nt) return set_err(c, MK_ERR_INVALID_ARG, "eps out of range");
      if ((int)value != c->eps)
        if (int rc = end_run(c, "MK_OPT_EPS_SAMPLES")) return rc;  // the window table of a run in progress would be stale
      c->eps = (int)value;
      return MK_OK;
    case MK_OPT_REGIME:
      if (value < 0 || value > 3 || value != std::floor(value)) return set_err(c, MK_ERR_INVALID_ARG, "regime must be 0..3");
      if ((int)value == 3 && !tc_supported(c)) return set_err(c, MK_ERR_INVALID_ARG, "tcgen05 3xTF32 regime needs an sm_100 device");
      c->regime = (int)value;
      return MK_OK;
    case MK_OPT_TIMING:
      if (value < 0 || value != std::floor(value) || value > 65536) return set_err(c, MK_ERR_INVALID_ARG, "MK_OPT_TIMING: 0 (off) or a stride 1 .. 65536");
      c->timing = (int)value;
      return MK_OK;
    case MK_OPT_FUSED_FINALS:
      c->fused_finals = value != 0.0;
      return MK_OK;
    case MK_OPT_RHAT_FORMAT: {
      if (value != 0.0 && value != 1.0) return set_err(c, MK_ERR_INVALID_ARG, "R^ format must be 0 (complex64) or 1 (q16 block float)");
      if ((int)value == c->rhat_format) return MK_OK;
      if (c->shots_loaded > 0) return set_err(c, MK_ERR_STATE, "MK_OPT_RHAT_FORMAT after mk_load_R: R^ is converted at ingest");
      if (c->nrow != c->n || c->nres != c->nrow || c->rhat_layout != 0) return set_err(c, MK_ERR_STATE, "compressed R^ is not available on row-sharded, streamed or tiled contexts");
      if (int rc = end_run(c, "MK_OPT_RHAT_FORMAT")) return rc;
      const size_t cnt = (size_t)c->n * c->nb * c->ld;
      if ((int)value == 1) {
        size_t cap = cnt;
        release(c, &c->d_Rhat, &cap);
        size_t cq = 0, cs = 0;
        if (int rc = ensure(c, &c->d_Rq, &cq, cnt, "Rhat q16")) return rc;
        if (int rc = ensure(c, &c->d_Rscale, &cs, cnt / 16, "Rhat scales")) return rc;
        if (int rc = check_cuda(c, cudaMemset(c->d_Rq, 0, cnt * sizeof(uint32_t)), "memset")) return rc;
        if (int rc = check_cuda(c, cudaMemset(c->d_Rscale, 0, cnt / 16 * sizeof(float)), "memset")) return rc;
      } else {
        size_t cq = cnt, cs = cnt / 16, cap = 0;
        release(c, &c->d_Rq, &cq);
        release(c, &c->d_Rscale, &cs);
        release(c, &c->d_qstage, &c->cap_qstage);
        if (int rc = ensure(c, &c->d_Rhat, &cap, cnt, "Rhat")) return rc;
        if (int rc = check_cuda(c, cudaMemset(c->d_Rhat, 0, cnt * sizeof(float2)), "memset")) return rc;
      }
      c->rhat_format = (int)value;
      return MK_OK;
    }
    case MK_OPT_RHAT_LAYOUT: {
      if (value != 0.0 && value != 1.0) return set_err(c, MK_ERR_INVALID_ARG, "R^ layout must be 0 (row-major) or 1 (tiled)");
      if ((int)value == c->rhat_layout) return MK_OK;
      if (c->shots_loaded > 0) return set_err(c, MK_ERR_STATE, "MK_OPT_RHAT_LAYOUT after mk_load_R: R^ is laid out at ingest");
      if (c->nrow != c->n || c->nres != c->nrow || c->rhat_format != 0)
        return set_err(c, MK_ERR_STATE, "tiled R^ is not available on row-sharded, streamed or compressed contexts");
      if ((int)value == 1 && !tc_supported(c)) return set_err(c, MK_ERR_INVALID_ARG, "tiled R^ needs the tcgen05 regime (an sm_100 device)");
      if (int rc = end_run(c, "MK_OPT_RHAT_LAYOUT")) return rc;
      const size_t rows = (int)value == 1 ? (size_t)((c->n + 127) / 128) * 128 : (size_t)c->n;  // receiver rows padded to whole tiles
      const size_t cnt = rows * c->nb * c->ld;
      size_t cap = 0;
      release(c, &c->d_Rhat, &cap);
      c->device_bytes -= (size_t)c->rhat_rows_alloc * c->nb * c->ld * sizeof(float2);
      if (int rc = ensure(c, &c->d_Rhat, &cap, cnt, "Rhat")) return rc;
      if (int rc = check_cuda(c, cudaMemset(c->d_Rhat, 0, cnt * sizeof(float2)), "memset")) return rc;
      c->rhat_rows_alloc = (int)rows;
      c->rhat_layout = (int)value;
      return MK_OK;
    }
    case MK_OPT_TUNE:
      if (value < 0 || value != std::floor(value) || value > 65535) return set_err(c, MK_ERR_INVALID_ARG, "tune mask out of range");
      c->tune = (int)value;
      return MK_OK;
    case MK_OPT_FFT_PATH:
      if (value < 0 || value > 2 || value != std::floor(value)) return set_err(c, MK_ERR_INVALID_ARG, "fft path must be 0..2");
      if ((int)value == 2 && c->nt != 2048 && c->nt != 4096)
        return set_err(c, MK_ERR_INVALID_ARG, "the register-resident transform path needs nt = 2048 or 4096");
      c->fft_path = (int)value;
      return MK_OK;
    default:
      return set_err(c, MK_ERR_INVALID_ARG, "unknown option");
  }
}

int mk_set_geometry(mk_ctx* c, const int* h_rec_of_shot, const float* h_weights) {
  MK_GUARD(c);
  if (c->nrow != c->n) return set_err(c, MK_ERR_STATE, "row-sharded context: mk_set_geometry is not available");
  if (c->shots_loaded > 0) return set_err(c, MK_ERR_STATE, "mk_set_geometry after mk_load_R: the weights are folded into R^ at ingest");
  if (int rc = end_run(c, "mk_set_geometry")) return rc;
  c->operand_key[0] = c->operand_key[1] = 0;  // rows that had a source may lose it: the operands are zeroed again
  c->custom_geometry = h_rec_of_shot || h_weights;
  return upload_geometry(c, h_rec_of_shot, h_weights);
}

int mk_get_info(mk_ctx* c, int key, double* value) {
  MK_GUARD(c);
  if (!value) return MK_ERR_INVALID_ARG;
  switch (key) {
    case MK_INFO_NB: *value = c->nb; return MK_OK;
    case MK_INFO_KLO: *value = c->klo; return MK_OK;
    case MK_INFO_KHI: *value = c->khi; return MK_OK;
    case MK_INFO_RHAT_BYTES: *value = 8.0 * c->nrow * (double)c->nb * c->ns; return MK_OK;
    case MK_INFO_RHAT_BYTES_PADDED: *value = 8.0 * c->nrow * (double)c->nb * c->ld; return MK_OK;
    case MK_INFO_RHAT_BYTES_STORED: *value = (c->rhat_format == 1 ? 4.25 : 8.0) * c->nrow * (double)c->nb * c->ld; return MK_OK;
    case MK_INFO_LD_SHOT: *value = c->ld; return MK_OK;
    case MK_INFO_SHOTS_LOADED: *value = c->shots_loaded; return MK_OK;
    case MK_INFO_SYN_LAUNCHES: *value = (double)(c->ev_used / 2); return MK_OK;
    case MK_INFO_SYN_MS_TOTAL: {
      if (int rc = check_cuda(c, cudaStreamSynchronize(c->stream), "cudaStreamSynchronize")) return rc;
      double tot = 0.0;
      for (size_t i = 0; i + 1 < c->ev_used; i += 2) {
        float ms = 0.f;
        if (int rc = check_cuda(c, cudaEventElapsedTime(&ms, c->ev[i], c->ev[i + 1]), "cudaEventElapsedTime")) return rc;
        tot += ms;
      }
      *value = tot;
      return MK_OK;
    }
    case MK_INFO_SYN_RESET: c->ev_used = 0; c->syn_count = 0; *value = 0; return MK_OK;
    case MK_INFO_SYN_COUNT: *value = (double)c->syn_count; return MK_OK;
    case MK_INFO_KERNEL_LAUNCHES: *value = (double)c->launches; return MK_OK;
    case MK_INFO_REGIME_USED: *value = c->last_regime; return MK_OK;
    case MK_INFO_DEVICE_BYTES: *value = (double)c->device_bytes; return MK_OK;
    case MK_INFO_RESIDENT_ROWS: *value = c->nres; return MK_OK;
    case MK_INFO_WINDOW_ROWS: *value = c->win_rows; return MK_OK;
    case MK_INFO_H2D_BYTES: *value = c->h2d_bytes; return MK_OK;
    case MK_INFO_RHAT_LAYOUT: *value = c->rhat_layout; return MK_OK;
    default: return set_err(c, MK_ERR_INVALID_ARG, "unknown info key");
  }
}

int mk_load_R(mk_ctx* c, const float* d_R_time, int shot0, int nshots) {
  MK_GUARD(c);
  if (!d_R_time || shot0 < 0 || nshots <= 0 || shot0 + nshots > c->ns) return set_err(c, MK_ERR_INVALID_ARG, "mk_load_R: bad shot range");
  if (int rc = end_run(c, "mk_load_R")) return rc;  // a run in progress was started from another R^: it is over
  if (c->rhat_format == 1) {
    // compressed R^: whole 16-shot blocks only (a block's scale needs all of its shots); sub-chunks of <= 64 shots go
    // through an fp32 stage [n * nb][<= 64] and the quantiser
    if (shot0 % 16 != 0 || (nshots % 16 != 0 && shot0 + nshots != c->ns))
      return set_err(c, MK_ERR_INVALID_ARG, "mk_load_R with compressed R^: shot0 and nshots must be multiples of 16 (except at the last shot)");
    const size_t rows = (size_t)c->n * c->nb;
    if (int rc = ensure(c, &c->d_qstage, &c->cap_qstage, rows * 64, "q16 stage")) return rc;
    for (int s0 = 0; s0 < nshots; s0 += 64) {
      const int m = std::min(64, nshots - s0), ldc = ((m + 15) / 16) * 16;
      if (m != ldc)
        if (int rc = check_cuda(c, cudaMemsetAsync(c->d_qstage, 0, rows * ldc * sizeof(float2), c->stream), "memset q16 stage")) return rc;
      RowBlock rb{c->d_qstage - (shot0 + s0), 0, c->n, ldc};  // the ingest kernel addresses columns by global shot index
      if (int rc = launch_load_R(c, rb, d_R_time + (size_t)s0 * c->n * c->nt, shot0 + s0, m)) return rc;
      if (int rc = launch_quantize_q16(c, c->d_qstage, ldc, shot0 + s0)) return rc;
    }
  } else if (c->nres > 0)
    if (int rc = launch_load_R(c, RowBlock{c->d_Rhat, c->r0, c->nres}, d_R_time, shot0, nshots)) return rc;
  if (c->nres < c->nrow) {  // out-of-core rows: the ingest kernel writes them to the mapped host memory directly
    if (int rc = launch_load_R(c, RowBlock{c->h_Rhat_dev, c->nres, c->nrow - c->nres}, d_R_time, shot0, nshots)) return rc;
    c->win_block[0] = c->win_block[1] = -1;  // what the windows hold is stale
  }
  for (int s = shot0; s < shot0 + nshots; ++s)
    if (!c->shot_loaded[s]) {
      c->shot_loaded[s] = 1;
      ++c->shots_loaded;
    }
  return MK_OK;
}

int mk_load_R_rows(mk_ctx* c, const float* d_R_rows, int shot0, int nshots) {
  MK_GUARD(c);
  if (!d_R_rows || shot0 < 0 || nshots <= 0 || shot0 + nshots > c->ns) return set_err(c, MK_ERR_INVALID_ARG, "mk_load_R_rows: bad shot range");
  if (c->rhat_format == 1 || c->nres < c->nrow) return set_err(c, MK_ERR_STATE, "mk_load_R_rows: not available with compressed or out-of-core R^");
  if (int rc = end_run(c, "mk_load_R_rows")) return rc;
  // the kernels address the source by the global receiver index: shift the base so that row r0 is the array's first
  RowBlock rb{c->d_Rhat, c->r0, c->nrow};
  rb.src_n = c->nrow;
  if (int rc = launch_load_R(c, rb, d_R_rows - (ptrdiff_t)c->r0 * c->nt, shot0, nshots)) return rc;
  for (int s = shot0; s < shot0 + nshots; ++s)
    if (!c->shot_loaded[s]) {
      c->shot_loaded[s] = 1;
      ++c->shots_loaded;
    }
  return MK_OK;
}

int mk_load_R_host(mk_ctx* c, const float* h_R_time, int shot0, int nshots) {
  MK_GUARD(c);
  if (!h_R_time || shot0 < 0 || nshots <= 0 || shot0 + nshots > c->ns) return set_err(c, MK_ERR_INVALID_ARG, "mk_load_R_host: bad shot range");
  const size_t per_shot = (size_t)c->n * c->nt;
  size_t chunk = ((size_t)1 << 28) / per_shot;  // <= 1 GiB of fp32 per staging chunk
  if (chunk < 1) chunk = 1;
  if (chunk > (size_t)nshots) chunk = nshots;
  if (int rc = ensure(c, &c->d_stage, &c->cap_stage, chunk * per_shot, "staging")) return rc;
  for (int s = 0; s < nshots; s += (int)chunk) {
    const int ns = std::min((int)chunk, nshots - s);
    if (int rc = check_cuda(c, cudaMemcpyAsync(c->d_stage, h_R_time + (size_t)s * per_shot, ns * per_shot * sizeof(float),
                                               cudaMemcpyHostToDevice, c->stream), "H2D R chunk")) return rc;
    if (int rc = mk_load_R(c, c->d_stage, shot0 + s, ns)) return rc;
  }
  return check_cuda(c, cudaStreamSynchronize(c->stream), "cudaStreamSynchronize");
}

// a1.  ext_plus / ext_min: caller-owned [nfoc][nrec][nt] buffers to accumulate f1plus / f1min in (mk_run hands its output
// fields in, which saves the copies at the end and the library's own fields), or NULL for the library's own.
static int begin_impl(mk_ctx* c, const float* d_Gd, const float* d_td, int nfoc, float* ext_plus, float* ext_min) {
  MK_GUARD(c);
  if (!d_Gd || !d_td || nfoc <= 0) return set_err(c, MK_ERR_INVALID_ARG, "mk_begin: bad arguments");
  if (c->shots_loaded != c->ns) return set_err(c, MK_ERR_STATE, "mk_begin before every shot of R was loaded");
  int regime = 0;
  if (int rc = resolve_regime(c, nfoc, &regime)) return rc;
  const int ldf = ldf_for(regime, nfoc);
  const size_t ntime = (size_t)nfoc * c->n * c->nt;
  const size_t nS = (size_t)c->n * c->nb * ldf;
  c->begun = false;
  {
    if (!ext_plus)
      if (int rc = ensure(c, &c->d_f1plus, &c->cap_time, ntime, "f1plus")) return rc;
    if (!ext_min)
      if (int rc = ensure(c, &c->d_f1min, &c->cap_time_min, ntime, "f1min")) return rc;
    c->acc_plus = ext_plus ? ext_plus : c->d_f1plus;
    c->acc_min = ext_min ? ext_min : c->d_f1min;
    size_t capS = c->cap_Shat;
    if (int rc = ensure(c, &c->d_Shat, &c->cap_Shat, nS, "Shat")) return rc;
    if (int rc = ensure(c, &c->d_phat, &capS, nS, "phat")) return rc;
    if (int rc = ensure(c, &c->d_h, &c->cap_h, (size_t)nfoc * c->n, "window table")) return rc;
  }
  c->nfoc = nfoc;
  c->ldf = ldf;
  c->run_regime = regime;
  c->iter = 0;
  c->contracted = false;
  c->prepared_field = 0;
  if (int rc = prepare_operand(c, 0, nfoc, ldf)) return rc;
  if (int rc = check_cuda(c, cudaMemsetAsync(c->d_phat, 0, nS * sizeof(float2), c->stream), "memset phat")) return rc;
  if (int rc = check_cuda(c, cudaMemsetAsync(c->acc_min, 0, ntime * sizeof(float), c->stream), "memset f1min")) return rc;
  if (int rc = launch_window(c, d_td, c->d_h, nfoc * c->n)) return rc;
  // a1: N_{-1} = f1plus = T G_d; N^_{-1} = conj(G_d^)     [PAPER.md:19, 67, 74-75]
  if (int rc = check_peers(c, 0)) return rc;
  const bool sharded = c->nrow != c->n;
  if (sharded)  // the rows of other ranks stay zero in this rank's fields
    if (int rc = check_cuda(c, cudaMemsetAsync(c->acc_plus, 0, ntime * sizeof(float), c->stream), "memset f1plus")) return rc;
  if (int rc = launch_fwd(c, d_Gd, operand_out(c, 0, ldf), nfoc, /*conj_out=*/true, c->acc_plus)) return rc;
  c->operand_stale[0] = sharded;
  c->begun = true;
  return MK_OK;
}

int mk_begin(mk_ctx* c, const float* d_Gd, const float* d_td, int nfoc) { return begin_impl(c, d_Gd, d_td, nfoc, nullptr, nullptr); }

int mk_step_contract(mk_ctx* c) {
  MK_GUARD(c);
  if (!c->begun) return set_err(c, MK_ERR_STATE, "mk_step before mk_begin");
  if (c->contracted) return set_err(c, MK_ERR_STATE, "mk_step_contract twice without mk_step_post");
  if (int rc = contract(c, 0, c->d_Shat, c->nfoc, c->ldf, c->run_regime)) return rc;                       // a2  [PAPER.md:69]
  c->contracted = true;
  return MK_OK;
}

int mk_step_post(mk_ctx* c, float* d_N_i) {
  MK_GUARD(c);
  if (!c->begun || !c->contracted) return set_err(c, MK_ERR_STATE, "mk_step_post without mk_step_contract");
  if (int rc = check_peers(c, 0)) return rc;
  if (int rc = launch_post(c, operand_out(c, 0, c->ldf), (c->iter % 2) == 0, d_N_i)) return rc;     // a3..a6
  c->operand_stale[0] = c->nrow != c->n;
  c->contracted = false;
  ++c->iter;
  return MK_OK;
}

int mk_step(mk_ctx* c, float* d_N_i) {
  if (int rc = mk_step_contract(c)) return rc;
  return mk_step_post(c, d_N_i);
}

static int scratch_operands(mk_ctx* c, int nfoc, int ldf) {
  const size_t nS = (size_t)c->n * c->nb * ldf;
  if (int rc = ensure(c, &c->d_Shat2, &c->cap_Shat2, nS, "Shat scratch")) return rc;
  return prepare_operand(c, 1, nfoc, ldf);
}

int mk_finish(mk_ctx* c, const mk_outputs* o) {
  MK_GUARD(c);
  if (!c->begun) return set_err(c, MK_ERR_STATE, "mk_finish before mk_begin");
  if (!o) return set_err(c, MK_ERR_INVALID_ARG, "mk_finish: null outputs");
  if (o->N_last) return set_err(c, MK_ERR_INVALID_ARG, "N_last is delivered by mk_run (or by mk_step's d_N_i), not by mk_finish");
  const size_t bytes = (size_t)c->nfoc * c->n * c->nt * sizeof(float);
  if (int rc = check_output_alias(c, o, c->acc_plus, c->acc_min, bytes)) return rc;
  if ((o->f1plus && o->f1plus != c->acc_plus && (overlaps(o->f1plus, c->acc_plus, bytes) || overlaps(o->f1plus, c->acc_min, bytes))) ||
      (o->f1min && o->f1min != c->acc_min && (overlaps(o->f1min, c->acc_plus, bytes) || overlaps(o->f1min, c->acc_min, bytes))) ||
      (o->f1plus && overlaps(o->f1plus, o->f1min, bytes)))
    return set_err(c, MK_ERR_INVALID_ARG, "mk_finish: the f1plus / f1min outputs overlap each other or the accumulators");
  if (o->f1plus && o->f1plus != c->acc_plus)  // mk_run accumulates in the caller's field directly
    if (int rc = check_cuda(c, cudaMemcpyAsync(o->f1plus, c->acc_plus, bytes, cudaMemcpyDeviceToDevice, c->stream), "copy f1plus")) return rc;
  if (o->f1min && o->f1min != c->acc_min)
    if (int rc = check_cuda(c, cudaMemcpyAsync(o->f1min, c->acc_min, bytes, cudaMemcpyDeviceToDevice, c->stream), "copy f1min")) return rc;
  if ((o->Gminus || o->Gplus) && c->nrow != c->n)
    return set_err(c, MK_ERR_STATE, "row-sharded context: G^- / G^+ need mk_finish_prepare, an exchange of slot 1, mk_finish_complete");
  // Few focal points: the two extra syntheses of the finals ("estimating each component requires an extra
  // synthesis") are ONE pass over R^ with 2 nfoc right-hand sides — columns [0, nfoc) = spectrum of f1plus (G^-),
  // [nfoc, 2 nfoc) = spectrum of T f1min (G^+) — in the bandwidth-bound regime that costs little more than one.
  const bool fuse = o->Gminus && o->Gplus && c->fused_finals && c->run_regime == 1 && (c->nfoc == 1 || c->nfoc == 2 || c->nfoc == 4) &&
                    gemv_supported(c, 2 * c->nfoc);
  if (fuse) {
    const int nf = c->nfoc, ldf2 = 2 * nf;
    if (int rc = ensure(c, &c->d_Shat2, &c->cap_Shat2, (size_t)c->n * c->nb * ldf2, "Shat scratch")) return rc;
    if (int rc = prepare_operand(c, 1, ldf2, ldf2)) return rc;
    OperandOut O = operand_out(c, 1, ldf2);
    if (int rc = launch_fwd(c, c->acc_plus, O, nf, false, nullptr)) return rc;
    O.plain += nf;
    if (int rc = launch_fwd(c, c->acc_min, O, nf, true, nullptr)) return rc;
    if (int rc = contract(c, 1, c->d_Shat2, ldf2, ldf2, 1)) return rc;
    if (int rc = launch_inv(c, c->d_Shat2, nf, ldf2, o->Gminus, 1.f, c->acc_min, -1.f, nullptr, 0.f)) return rc;       // [PAPER.md:87-88]
    if (int rc = launch_inv(c, c->d_Shat2 + nf, nf, ldf2, o->Gplus, -1.f, nullptr, 0.f, c->acc_plus, 1.f)) return rc;   // [G4]
  } else if (o->Gminus) {
    if (int rc = mk_finish_prepare(c, MK_FIELD_GMINUS)) return rc;
    if (int rc = mk_finish_complete(c, MK_FIELD_GMINUS, o->Gminus)) return rc;
  }
  if (!fuse && o->Gplus) {
    if (int rc = mk_finish_prepare(c, MK_FIELD_GPLUS)) return rc;
    if (int rc = mk_finish_complete(c, MK_FIELD_GPLUS, o->Gplus)) return rc;
  }
  if (o->G) {  // G = p^- + T f2 = p^- + T f1plus - f1min   [PAPER.md:24; G3]
    if (int rc = launch_inv(c, c->d_phat, c->nfoc, c->ldf, o->G, 1.f, c->acc_min, -1.f, c->acc_plus, 1.f)) return rc;
  }
  return MK_OK;
}

int mk_finish_prepare(mk_ctx* c, int field) {
  MK_GUARD(c);
  if (!c->begun) return set_err(c, MK_ERR_STATE, "mk_finish_prepare before mk_begin");
  if (field != MK_FIELD_GMINUS && field != MK_FIELD_GPLUS) return set_err(c, MK_ERR_INVALID_ARG, "mk_finish_prepare: unknown field");
  if (int rc = scratch_operands(c, c->nfoc, c->ldf)) return rc;
  // G^- = R f1plus - f1min [PAPER.md:87-88; G5]: operand = spectrum of f1plus;  G^+ = T f1plus - R (T f1min) [PAPER.md:24; G4]:
  // operand = spectrum of T f1min = conj of the spectrum of f1min
  if (int rc = check_peers(c, 1)) return rc;
  const bool minus = field == MK_FIELD_GMINUS;
  if (int rc = launch_fwd(c, minus ? c->acc_plus : c->acc_min, operand_out(c, 1, c->ldf), c->nfoc, !minus, nullptr)) return rc;
  c->operand_stale[1] = c->nrow != c->n;
  c->prepared_field = field;
  return MK_OK;
}

int mk_finish_complete(mk_ctx* c, int field, float* d_out) {
  MK_GUARD(c);
  if (!d_out) return set_err(c, MK_ERR_INVALID_ARG, "mk_finish_complete: null output");
  if (!c->begun || c->prepared_field != field || field == 0) return set_err(c, MK_ERR_STATE, "mk_finish_complete without the matching mk_finish_prepare");
  const int regime = c->run_regime;
  if (int rc = contract(c, 1, c->d_Shat2, c->nfoc, c->ldf, regime)) return rc;
  c->prepared_field = 0;
  if (field == MK_FIELD_GMINUS) return launch_inv(c, c->d_Shat2, c->nfoc, c->ldf, d_out, 1.f, c->acc_min, -1.f, nullptr, 0.f);
  return launch_inv(c, c->d_Shat2, c->nfoc, c->ldf, d_out, -1.f, nullptr, 0.f, c->acc_plus, 1.f);
}

int mk_operand(mk_ctx* c, int slot, mk_operand_view* v) {
  MK_GUARD(c);
  if (!v || slot < 0 || slot > 1) return set_err(c, MK_ERR_INVALID_ARG, "mk_operand: bad arguments");
  if (!c->begun && !c->reserved) return set_err(c, MK_ERR_STATE, "mk_operand before mk_begin / mk_operand_reserve");
  std::memset(v, 0, sizeof *v);
  v->nb = c->nb;
  v->row0 = c->r0;
  v->nrows = c->nrow;
  v->nplanes = 1;  // every regime reads the one complex operand N^[k][s][f] (interleaved floats)
  v->plane[0] = reinterpret_cast<float*>(slot ? c->d_Nhat2 : c->d_Nhat);
  v->rows_per_bin = c->ld;
  v->rows_per_rec = 1;
  v->row_floats = 2 * c->ldf;
  if (!v->plane[0]) return set_err(c, MK_ERR_STATE, "mk_operand: this slot has no operand yet");
  return MK_OK;
}

int mk_operand_exchanged(mk_ctx* c, int slot) {
  MK_GUARD(c);
  if (slot < 0 || slot > 1) return set_err(c, MK_ERR_INVALID_ARG, "mk_operand_exchanged: bad slot");
  c->operand_stale[slot] = false;
  return MK_OK;
}

int mk_ipc_export(const void* d_ptr, unsigned char handle[64]) {
  static_assert(sizeof(cudaIpcMemHandle_t) == 64, "CUDA IPC handle size");
  if (!d_ptr || !handle) return MK_ERR_INVALID_ARG;
  cudaIpcMemHandle_t h;
  if (cudaIpcGetMemHandle(&h, const_cast<void*>(d_ptr)) != cudaSuccess) {
    cudaGetLastError();
    return MK_ERR_CUDA;
  }
  std::memcpy(handle, &h, 64);
  return MK_OK;
}

int mk_ipc_open(const unsigned char handle[64], void** d_ptr) {
  if (!handle || !d_ptr) return MK_ERR_INVALID_ARG;
  cudaIpcMemHandle_t h;
  std::memcpy(&h, handle, 64);
  if (cudaIpcOpenMemHandle(d_ptr, h, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) {
    cudaGetLastError();
    *d_ptr = nullptr;
    return MK_ERR_CUDA;
  }
  return MK_OK;
}

int mk_ipc_close(void* d_ptr) {
  if (!d_ptr) return MK_OK;
  if (cudaIpcCloseMemHandle(d_ptr) != cudaSuccess) {
    cudaGetLastError();
    return MK_ERR_CUDA;
  }
  return MK_OK;
}

int mk_sync_create(mk_ctx* c, int rank, int world) {
  MK_GUARD(c);
  if (world < 1 || world > 8 || rank < 0 || rank >= world) return set_err(c, MK_ERR_INVALID_ARG, "mk_sync_create: need 0 <= rank < world <= 8");
  if (!c->write32_fn) {
    cudaDriverEntryPointQueryResult q;
    void* w = nullptr;
    void* t = nullptr;
    if (cudaGetDriverEntryPoint("cuStreamWriteValue32", &w, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess || !w ||
        cudaGetDriverEntryPoint("cuStreamWaitValue32", &t, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess || !t) {
      cudaGetLastError();
      return set_err(c, MK_ERR_CUDA, "stream memory operations (cuStreamWriteValue32 / cuStreamWaitValue32) are not available");
    }
    c->write32_fn = w;
    c->wait32_fn = t;
  }
  if (!c->d_sync_flags)
    if (int rc = check_cuda(c, cudaMalloc(&c->d_sync_flags, 8 * sizeof(uint32_t)), "cudaMalloc sync flags")) return rc;
  if (int rc = check_cuda(c, cudaMemset(c->d_sync_flags, 0, 8 * sizeof(uint32_t)), "memset sync flags")) return rc;
  c->sync_rank = rank;
  c->sync_world = world;
  c->sync_epoch = 0;
  c->sync_attached = world == 1;
  for (auto& p : c->sync_peer) p = nullptr;
  c->sync_peer[rank] = c->d_sync_flags;
  return MK_OK;
}

int mk_sync_flags(mk_ctx* c, void** d_flags) {
  MK_GUARD(c);
  if (!d_flags) return MK_ERR_INVALID_ARG;
  if (!c->d_sync_flags) return set_err(c, MK_ERR_STATE, "mk_sync_flags before mk_sync_create");
  *d_flags = c->d_sync_flags;
  return MK_OK;
}

int mk_sync_attach(mk_ctx* c, void* const* d_flags_of_rank) {
  MK_GUARD(c);
  if (!c->d_sync_flags) return set_err(c, MK_ERR_STATE, "mk_sync_attach before mk_sync_create");
  if (!d_flags_of_rank) return MK_ERR_INVALID_ARG;
  for (int g = 0; g < c->sync_world; ++g) {
    if (g == c->sync_rank) continue;
    if (!d_flags_of_rank[g]) return set_err(c, MK_ERR_INVALID_ARG, "mk_sync_attach: a peer's flag array is NULL");
    c->sync_peer[g] = static_cast<uint32_t*>(d_flags_of_rank[g]);
  }
  c->sync_attached = true;
  return MK_OK;
}

int mk_sync_barrier(mk_ctx* c) {
  MK_GUARD(c);
  if (!c->sync_attached) return set_err(c, MK_ERR_STATE, "mk_sync_barrier before mk_sync_create / mk_sync_attach");
  typedef CUresult (*Write32)(CUstream, CUdeviceptr, cuuint32_t, unsigned int);
  typedef CUresult (*Wait32)(CUstream, CUdeviceptr, cuuint32_t, unsigned int);
  const Write32 wr = reinterpret_cast<Write32>(c->write32_fn);
  const Wait32 wt = reinterpret_cast<Wait32>(c->wait32_fn);
  const uint32_t e = ++c->sync_epoch;
  CUstream st = reinterpret_cast<CUstream>(c->stream);
  for (int g = 0; g < c->sync_world; ++g) {
    if (g == c->sync_rank) continue;
    if (wr(st, reinterpret_cast<CUdeviceptr>(c->sync_peer[g] + c->sync_rank), e, CU_STREAM_WRITE_VALUE_DEFAULT) != CUDA_SUCCESS)
      return set_err(c, MK_ERR_CUDA, "cuStreamWriteValue32 failed");
  }
  for (int g = 0; g < c->sync_world; ++g) {
    if (g == c->sync_rank) continue;
    if (wt(st, reinterpret_cast<CUdeviceptr>(c->d_sync_flags + g), e, CU_STREAM_WAIT_VALUE_GEQ) != CUDA_SUCCESS)
      return set_err(c, MK_ERR_CUDA, "cuStreamWaitValue32 failed");
  }
  return MK_OK;
}

int mk_operand_reserve(mk_ctx* c, int nfoc) {
  MK_GUARD(c);
  if (nfoc <= 0) return set_err(c, MK_ERR_INVALID_ARG, "mk_operand_reserve: bad nfoc");
  int regime = 0;
  if (int rc = resolve_regime(c, nfoc, &regime)) return rc;
  const int ldf = ldf_for(regime, nfoc);
  if (c->begun && (nfoc != c->nfoc || regime != c->run_regime))  // another operand layout: the run in progress is over
    if (int rc = end_run(c, "mk_operand_reserve")) return rc;
  if (int rc = prepare_operand(c, 0, nfoc, ldf)) return rc;
  if (int rc = prepare_operand(c, 1, nfoc, ldf)) return rc;
  c->nfoc = nfoc;
  c->ldf = ldf;
  c->run_regime = regime;
  c->reserved = true;
  return MK_OK;
}

int mk_operand_attach(mk_ctx* c, int slot, int npeers, const mk_operand_view* peers) {
  MK_GUARD(c);
  if (slot < 0 || slot > 1 || npeers < 0 || npeers > kMaxPeers || (npeers > 0 && !peers))
    return set_err(c, MK_ERR_INVALID_ARG, "mk_operand_attach: bad arguments");
  c->npeer[slot] = 0;
  if (npeers == 0) return MK_OK;
  mk_operand_view mine;
  if (int rc = mk_operand(c, slot, &mine)) return rc;
  for (int p = 0; p < npeers; ++p) {
    const mk_operand_view& v = peers[p];
    if (v.nplanes != mine.nplanes || v.nb != mine.nb || v.rows_per_bin != mine.rows_per_bin || v.rows_per_rec != mine.rows_per_rec ||
        v.row_floats != mine.row_floats || !v.plane[0] || (v.nplanes == 2 && !v.plane[1]))
      return set_err(c, MK_ERR_INVALID_ARG, "mk_operand_attach: a peer's operand has another layout");
    c->peer_plane[slot][p] = v.plane[0];
  }
  c->npeer[slot] = npeers;
  c->peer_key[slot] = c->operand_key[slot];
  return MK_OK;
}

int mk_run(mk_ctx* c, const float* d_Gd, const float* d_td, int nfoc, int niter, const mk_outputs* o) {
  MK_GUARD(c);
  if (c->nrow != c->n) return set_err(c, MK_ERR_STATE, "row-sharded context: drive mk_begin / mk_step / mk_finish_* with the exchanges in between");
  if (niter < 0 || !o) return set_err(c, MK_ERR_INVALID_ARG, "mk_run: bad arguments");
  if (o->N_last && niter == 0) return set_err(c, MK_ERR_INVALID_ARG, "N_last needs niter >= 1");
  if (!d_Gd || nfoc <= 0) return set_err(c, MK_ERR_INVALID_ARG, "mk_run: bad arguments");
  {
    const size_t bytes = (size_t)nfoc * c->n * c->nt * sizeof(float);
    if (overlaps(o->f1plus, o->f1min, bytes) || overlaps(o->f1plus, d_Gd, bytes) || overlaps(o->f1min, d_Gd, bytes))
      return set_err(c, MK_ERR_INVALID_ARG, "mk_run: f1plus / f1min must not overlap each other or G_d");
    // with no caller field the library's own accumulators are used; they cannot overlap caller memory
    if (int rc = check_output_alias(c, o, o->f1plus, o->f1min, bytes)) return rc;
  }
  if (int rc = begin_impl(c, d_Gd, d_td, nfoc, o->f1plus, o->f1min)) return rc;  // accumulate in the caller's fields
  for (int i = 0; i < niter; ++i)
    if (int rc = mk_step(c, i == niter - 1 ? o->N_last : nullptr)) return rc;
  mk_outputs rest = *o;
  rest.N_last = nullptr;
  return mk_finish(c, &rest);
}

int mk_run_host(mk_ctx* c, const float* h_Gd, const float* h_td, int nfoc, int niter, const mk_outputs* ho) {
  MK_GUARD(c);
  if (c->nrow != c->n) return set_err(c, MK_ERR_STATE, "row-sharded context: mk_run_host is not available");
  if (!h_Gd || !h_td || nfoc <= 0 || niter < 0 || !ho) return set_err(c, MK_ERR_INVALID_ARG, "mk_run_host: bad arguments");
  if (ho->N_last && niter == 0) return set_err(c, MK_ERR_INVALID_ARG, "N_last needs niter >= 1");
  const size_t ntime = (size_t)nfoc * c->n * c->nt, ntd = (size_t)nfoc * c->n;
  // Small runs get one staging field per output, and the device -> host copies go to a second stream so that they
  // overlap the finals' syntheses; big ones (> 256 MiB per field) share one staging field and stay on one stream.
  const bool overlap = ntime * sizeof(float) <= ((size_t)256 << 20);
  const int nstage = overlap ? 4 : 1;
  if (int rc = ensure(c, &c->d_stage, &c->cap_stage, nstage * ntime + ntd, "staging")) return rc;
  float* d_field = c->d_stage;
  float* d_td = c->d_stage + nstage * ntime;
  if (overlap && !c->copy_stream) {
    if (int rc = check_cuda(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking), "cudaStreamCreate")) return rc;
    if (int rc = check_cuda(c, cudaEventCreateWithFlags(&c->copy_ev, cudaEventDisableTiming), "cudaEventCreate")) return rc;
  }
  cudaStream_t cs = overlap ? c->copy_stream : c->stream;
  // everything enqueued on the main stream so far may be copied out on the copy stream
  auto hand_over = [&]() -> int {
    if (!overlap) return MK_OK;
    if (int rc = check_cuda(c, cudaEventRecord(c->copy_ev, c->stream), "cudaEventRecord")) return rc;
    return check_cuda(c, cudaStreamWaitEvent(cs, c->copy_ev, 0), "cudaStreamWaitEvent");
  };
  if (int rc = check_cuda(c, cudaMemcpyAsync(d_field, h_Gd, ntime * sizeof(float), cudaMemcpyHostToDevice, c->stream), "H2D G_d")) return rc;
  if (int rc = check_cuda(c, cudaMemcpyAsync(d_td, h_td, ntd * sizeof(float), cudaMemcpyHostToDevice, c->stream), "H2D t_d")) return rc;
  if (int rc = mk_begin(c, d_field, d_td, nfoc)) return rc;
  float* hosts[5] = {ho->f1plus, ho->f1min, ho->G, ho->Gplus, ho->Gminus};
  // Step i adds to f1min (i even) or to f1plus (i odd): the accumulator the LAST step does not touch is final one step
  // earlier, and its copy to the host overlaps that last step instead of waiting behind it.
  const int early = (niter >= 1 && overlap) ? ((niter - 1) % 2 == 0 ? 0 : 1) : -1;
  for (int i = 0; i < niter; ++i) {
    const bool last = i == niter - 1;
    if (last && early >= 0 && hosts[early]) {
      if (int rc = hand_over()) return rc;
      if (int rc = check_cuda(c, cudaMemcpyAsync(hosts[early], early == 0 ? c->acc_plus : c->acc_min, ntime * sizeof(float), cudaMemcpyDeviceToHost, cs), "D2H accumulator")) return rc;
    }
    if (int rc = mk_step(c, last && ho->N_last ? d_field : nullptr)) return rc;
  }
  if (int rc = hand_over()) return rc;
  if (ho->N_last)
    if (int rc = check_cuda(c, cudaMemcpyAsync(ho->N_last, d_field, ntime * sizeof(float), cudaMemcpyDeviceToHost, cs), "D2H N_last")) return rc;
  for (int i = 0; i < 5; ++i) {
    if (!hosts[i] || i == early) continue;
    if (i == 0 || i == 1) {  // accumulators go straight from the library's buffers (the finals only read them)
      const float* src = i == 0 ? c->acc_plus : c->acc_min;
      if (int rc = check_cuda(c, cudaMemcpyAsync(hosts[i], src, ntime * sizeof(float), cudaMemcpyDeviceToHost, cs), "D2H accumulator")) return rc;
      continue;
    }
    float* d_out = overlap ? d_field + (size_t)(i - 1) * ntime : d_field;  // fields 1..3 of the staging area; field 0 holds N_last
    mk_outputs one{};
    if (i == 2) one.G = d_out;
    if (i == 3) one.Gplus = d_out;
    if (i == 4) one.Gminus = d_out;
    const bool both = overlap && i == 3 && hosts[4];  // G^+ and G^- in one call: they may share one pass over R^
    if (both) one.Gminus = d_field + (size_t)3 * ntime;
    if (int rc = mk_finish(c, &one)) return rc;
    if (int rc = hand_over()) return rc;
    if (int rc = check_cuda(c, cudaMemcpyAsync(hosts[i], d_out, ntime * sizeof(float), cudaMemcpyDeviceToHost, cs), "D2H output")) return rc;
    if (both) {
      if (int rc = check_cuda(c, cudaMemcpyAsync(hosts[4], one.Gminus, ntime * sizeof(float), cudaMemcpyDeviceToHost, cs), "D2H output")) return rc;
      break;
    }
  }
  if (overlap)
    if (int rc = check_cuda(c, cudaStreamSynchronize(cs), "cudaStreamSynchronize")) return rc;
  return check_cuda(c, cudaStreamSynchronize(c->stream), "cudaStreamSynchronize");
}

int mk_synthesis(mk_ctx* c, const float* d_N_in, float* d_S_out, int nfoc) {
  MK_GUARD(c);
  if (c->nrow != c->n) return set_err(c, MK_ERR_STATE, "row-sharded context: mk_synthesis is not available");
  if (!d_N_in || !d_S_out || nfoc <= 0) return set_err(c, MK_ERR_INVALID_ARG, "mk_synthesis: bad arguments");
  if (c->shots_loaded != c->ns) return set_err(c, MK_ERR_STATE, "mk_synthesis before every shot of R was loaded");
  int regime = 0;
  if (int rc = resolve_regime(c, nfoc, &regime)) return rc;
  const int ldf = ldf_for(regime, nfoc);
  if (int rc = scratch_operands(c, nfoc, ldf)) return rc;
  if (int rc = launch_fwd(c, d_N_in, operand_out(c, 1, ldf), nfoc, false, nullptr)) return rc;   // a6
  if (int rc = contract(c, 1, c->d_Shat2, nfoc, ldf, regime)) return rc;                          // a2
  return launch_inv(c, c->d_Shat2, nfoc, ldf, d_S_out, 1.f, nullptr, 0.f, nullptr, 0.f);     // a3
}

int mk_image(mk_ctx* c, const float* d_Gminus, float* d_image) {
  MK_GUARD(c);
  if (!d_Gminus || !d_image) return set_err(c, MK_ERR_INVALID_ARG, "mk_image: bad arguments");
  if (!c->begun) return set_err(c, MK_ERR_STATE, "mk_image before a run");
  const float wm = (float)(c->dt * c->dx), we = (float)(c->dt * c->dx * 0.5);
  // enough CTAs to fill the machine several times over, whole receivers per CTA
  const long long traces = (long long)c->nfoc * c->n;
  int rows_per_cta = (int)std::max<long long>(1, traces / ((long long)c->num_sms * 16));
  rows_per_cta = std::min(rows_per_cta, c->n);
  const int nchunk = (c->n + rows_per_cta - 1) / rows_per_cta;
  if (int rc = ensure(c, &c->d_img_part, &c->cap_img_part, (size_t)c->nfoc * nchunk, "image partial sums")) return rc;
  k_image_partial<<<dim3(c->nfoc, nchunk), kImgThreads, 0, c->stream>>>(d_Gminus, c->acc_plus, c->d_img_part, c->n, c->nt, rows_per_cta, wm, we);
  ++c->launches;
  if (int rc = check_cuda(c, cudaGetLastError(), "k_image_partial")) return rc;
  k_image_final<<<(c->nfoc + 127) / 128, 128, 0, c->stream>>>(c->d_img_part, d_image, c->nfoc, nchunk);
  ++c->launches;
  return check_cuda(c, cudaGetLastError(), "k_image");
}

int mk_image_static(mk_ctx* c, const float* d_Gminus, const float* d_f1plus, float* d_image, int nfoc) {
  MK_GUARD(c);
  if (!d_Gminus || !d_f1plus || !d_image || nfoc <= 0) return set_err(c, MK_ERR_INVALID_ARG, "mk_image_static: bad arguments");
  const float wm = (float)(c->dt * c->dx), we = (float)(c->dt * c->dx * 0.5);
  // the same grid as mk_image (same partial sums in the same order: the two calls give the same bits)
  const long long traces = (long long)nfoc * c->n;
  int rows_per_cta = (int)std::max<long long>(1, traces / ((long long)c->num_sms * 16));
  rows_per_cta = std::min(rows_per_cta, c->n);
  const int nchunk = (c->n + rows_per_cta - 1) / rows_per_cta;
  const long long nparts = (long long)nfoc * nchunk;
  if (nparts > MK_IMAGE_STATIC_MAX_PARTIALS) {
    char buf[224];
    snprintf(buf, sizeof buf,
             "mk_image_static: %d focal points x %d receiver chunks = %lld partial sums, the static scratch array holds "
             "MK_IMAGE_STATIC_MAX_PARTIALS = %d (use mk_image)", nfoc, nchunk, nparts, (int)MK_IMAGE_STATIC_MAX_PARTIALS);
    return set_err(c, MK_ERR_INVALID_ARG, buf);
  }
  double* part = nullptr;
  if (int rc = image_static_scratch(c, &part)) return rc;
  // nothing to clear: k_image_partial writes every one of the nparts sums before k_image_final reads them
  k_image_partial<<<dim3(nfoc, nchunk), kImgThreads, 0, c->stream>>>(d_Gminus, d_f1plus, part, c->n, c->nt, rows_per_cta, wm, we);
  ++c->launches;
  if (int rc = check_cuda(c, cudaGetLastError(), "k_image_partial (static scratch)")) return rc;
  k_image_final<<<(nfoc + 127) / 128, 128, 0, c->stream>>>(part, d_image, nfoc, nchunk);
  ++c->launches;
  return check_cuda(c, cudaGetLastError(), "k_image_final (static scratch)");
}

}  // extern "C"

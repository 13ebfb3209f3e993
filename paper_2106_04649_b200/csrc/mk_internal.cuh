// mk_internal.cuh — context and kernel launchers shared by the translation units of libmk (not part of the ABI).
#pragma once

#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/mk.h"
#include "fft_core.cuh"

// Device layouts (complex64 = float2, interleaved re/im):
// n = receivers (rows of R^, traces per focal point), ns = shots (the integration index; ns == n for a co-located spread)
//   Rhat [n][nb][ld]      R^[r][k][s] * dt * w[s]; ld = round_up(ns, 16); pad columns are zero       (a0)
//   Nhat [nb][ld][ldf]    N^[k][s][f]; pad rows (s >= n) and pad columns (f >= nfoc) are zero        (a1, a6)
//   (ldf = nfoc for the streaming GEMV, round_up(nfoc, 4) for the FFMA GEMM, round_up(nfoc, 16) for the tcgen05 GEMM,
//   whose TMA boxes are 32 floats wide; every regime reads this one operand)
//   Shat [n][nb][ldf]     S^[r][k][f]                                                                 (a2)
//   phat [n][nb][ldf]     running p^- spectrum                                                        (a3)
//   f1plus, f1min [nfoc][n][nt] fp32 time domain                                                      (a5)
//   h [nfoc][n] int32     window half-widths                                                          (a4)
struct mk_ctx {
  int n = 0, ns = 0, nt = 0, nb = 0, klo = 0, khi = 0, ld = 0;
  int r0 = 0, nrow = 0;  // receiver rows this context owns (row sharding; nrow == n: everything)
  bool operand_stale[2] = {false, false};  // sharded: rows produced locally but not yet exchanged
  int prepared_field = 0;                  // mk_finish_prepare
  double dt = 0, dx = 0, fmin = 0, fmax = 0;
  int eps = 8, regime = 0, timing = 0;
  cudaStream_t stream = nullptr;
  mkfft::Plan plan{};
  int num_sms = 0;
  size_t smem_optin = 0;

  float2* d_tw = nullptr;    // [nt] e^{-2 pi i k / nt}
  float2* d_tw1k = nullptr;  // [32][32] e^{-2 pi i k1 t / 1024}: middle twiddles of the register-resident path
  bool fused_finals = true;  // MK_OPT_FUSED_FINALS
  int fft_path = 0;          // MK_OPT_FFT_PATH: 0 auto, 1 generic shared-memory passes, 2 register-resident
  float2* d_Rhat = nullptr;  // [n][nb][ld]
  float* d_wscale = nullptr;      // [ns] dt * w[s]: folded into R^ at ingest (trapezoid over the shots unless mk_set_geometry)
  int* d_shot_of_rec = nullptr;   // [n] shot co-located with each receiver, -1 = none; nullptr = identity (co-located spread)
  bool custom_geometry = false;
  std::vector<unsigned char> shot_loaded;
  int shots_loaded = 0;
  // out-of-core R^ (mk_create_streamed): rows [0, nres) of R^ live in d_Rhat, rows [nres, nrow) in
  // pinned, device-mapped host memory and pass through two windows of win_rows rows in HBM during every contraction
  int nres = 0;                   // rows of R^ resident in HBM (== nrow unless streamed)
  float2* h_Rhat = nullptr;       // [(nrow - nres)][nb][ld], pinned + mapped (host address)
  float2* h_Rhat_dev = nullptr;   // the same memory as the ingest kernels address it
  int win_rows = 0;
  float2* d_win[2] = {nullptr, nullptr};
  int win_block[2] = {-1, -1};    // row block each window holds (-1: none)
  bool win_reverse = false;       // passes alternate direction, so the two blocks left in the windows are reused
  cudaStream_t h2d_stream = nullptr;
  cudaEvent_t win_ready[2] = {nullptr, nullptr}, win_free[2] = {nullptr, nullptr}, win_main = nullptr;
  double h2d_bytes = 0;           // bytes of R^ copied host -> device by contractions since creation
  // compressed R^ (MK_OPT_RHAT_FORMAT = 1, mk_syn_gemv_q16.cu): block floating point, int16 mantissas, one scale per 16 shots
  int rhat_format = 0;
  uint32_t* d_Rq = nullptr;       // [n][nb][ld] packed (re, im) int16
  float* d_Rscale = nullptr;      // [n][nb][ld / 16]
  float2* d_qstage = nullptr;     // fp32 spectra of one sub-chunk of shots on their way to the quantiser
  size_t cap_qstage = 0;

  // run state
  int nfoc = 0, ldf = 0, iter = 0;
  bool begun = false;
  bool contracted = false;  // mk_step_contract done, mk_step_post pending
  bool reserved = false;  // mk_operand_reserve: operands of c->nfoc exist
  float* d_f1plus = nullptr;
  float* d_f1min = nullptr;
  size_t cap_time = 0, cap_time_min = 0;  // capacities (floats) of d_f1plus / d_f1min
  float* acc_plus = nullptr;  // the accumulators of the current run: the library's own fields, or (mk_run) the caller's
  float* acc_min = nullptr;   // f1plus / f1min output fields
  float2* d_Nhat = nullptr;
  float2* d_Shat = nullptr;
  float2* d_phat = nullptr;
  size_t cap_Nhat = 0, cap_Shat = 0;  // capacities in float2
  int* d_h = nullptr;
  size_t cap_h = 0;
  // scratch operands for mk_synthesis / finals (so a run in progress is not disturbed)
  float2* d_Nhat2 = nullptr;
  float2* d_Shat2 = nullptr;
  size_t cap_Nhat2 = 0, cap_Shat2 = 0;
  long long operand_key[2] = {0, 0};   // layout the slot's operand was last zeroed for (0 = not zeroed)
  int npeer[2] = {0, 0};               // mk_operand_attach
  float* peer_plane[2][7] = {};        // [slot][peer]: the peers' operands of the same layout
  long long peer_key[2] = {0, 0};      // operand layout the peers were attached for
  // regime 3: cached TMA descriptors (CUtensorMap is 128 bytes, 64-byte aligned), built by mk_syn_tc.cu
  alignas(64) unsigned char tmap_A[3][128];  // [resident rows / window 0 / window 1]
  alignas(64) unsigned char tmap_B[2][128];  // [main / scratch operand]
  const void* tmap_A_key[3] = {nullptr, nullptr, nullptr};
  int tmap_A_rows[3] = {0, 0, 0};
  const void* tmap_B_key[2] = {nullptr, nullptr};
  int tmap_B_ldf[2] = {0, 0};
  uint32_t* d_tc_progress = nullptr;  // tcgen05 contraction: A boxes asked for, per CTA (sibling CTAs keep in step)
  // mk_sync_*: stream-ordered barrier between ranks
  uint32_t* d_sync_flags = nullptr;   // [sync_world] epochs the other ranks have written here
  uint32_t* sync_peer[8] = {};        // every rank's flag array as mapped in this process ([sync_rank] = own)
  int sync_rank = -1, sync_world = 0;
  uint32_t sync_epoch = 0;
  bool sync_attached = false;
  void* write32_fn = nullptr;         // cuStreamWriteValue32 / cuStreamWaitValue32, resolved through the runtime
  void* wait32_fn = nullptr;
  void* encode_fn = nullptr;  // cuTensorMapEncodeTiled, resolved at run time through the CUDA runtime
  float* d_stage = nullptr;  // host-call staging
  double* d_img_part = nullptr;  // mk_image: per (focal point, receiver chunk) partial sums
  size_t cap_img_part = 0;
  cudaStream_t copy_stream = nullptr;  // mk_run_host: device -> host copies overlapping the finals
  cudaEvent_t copy_ev = nullptr;
  size_t cap_stage = 0;

  size_t device_bytes = 0;
  long launches = 0;
  int run_regime = 0;   // regime of the run in progress / of the reserved operands: set by mk_begin and mk_operand_reserve only
  int last_regime = 0;  // regime of the last contraction launch (MK_INFO_REGIME_USED; information only)
  size_t smem_sm = 0;   // shared memory per SM
  int rhat_rows_alloc = 0;  // receiver rows d_Rhat was allocated for (tiled: padded to a multiple of 128)
  int rhat_layout = 0;  // MK_OPT_RHAT_LAYOUT: 0 row-major [rec][bin][shot], 1 tiled for the tensor regime
  int tune = 0;         // MK_OPT_TUNE: measurement switches (bit mask, include/mk.h)
  int dev = 0;          // CUDA device the context lives on (made current at the top of every entry point)

  // timing of contraction launches
  std::vector<cudaEvent_t> ev;  // pairs
  size_t ev_used = 0;
  size_t syn_count = 0;  // contraction launches since MK_INFO_SYN_RESET, timed or not

  std::string err;
  int sticky = 0;
};

namespace mk {

struct FftParams {
  mkfft::Plan plan;
  const float2* tw;
  const float* wscale;  // [ns] dt * w[s] (k_load_R)
  int n, nb, klo, ld, ldf, nfoc;
  int tiled;  // k_load_R: layout of R^ (rhat_index)
  int r0;  // first receiver row of this context (grid row b handles receiver r0 + b; R^ is stored from row r0 on)
};

// R^ element (receiver row rr of the block, bin kk, shot s) -> offset in float2.  Row-major (the default, what the streaming
// GEMV wants): [row][bin][ld].  Tiled (MK_OPT_RHAT_LAYOUT = 1, for the tensor regime): [row / 128][bin][shot / 16] boxes of
// [128 rows][16 shots] = 16 KB contiguous, the unit the tcgen05 contraction feeds on, stored already in the shared-memory
// layout its split warps read (the 16-byte chunk c = (s % 16) / 2 of row r sits at chunk position c ^ (r & 7)).
__host__ __device__ __forceinline__ size_t rhat_index(int tiled, int rr, int kk, int s, int nb, int ld) {
  if (!tiled) return ((size_t)rr * nb + kk) * ld + s;
  const int row = rr & 127, c = (s & 15) >> 1;
  return ((((size_t)(rr >> 7) * nb + kk) * (ld >> 4) + (s >> 4)) * 128 + row) * 16 + (size_t)(((c ^ (row & 7)) << 1) | (s & 1));
}

// Programmatic dependent launch (the chain of one iteration is launch-latency and drain bound when the focal points are few:
// 40 kernels of 3 .. 190 us per config-1 step).  A kernel launched through launch_pdl may be scheduled as soon as every CTA
// of the kernel in front of it on the stream has called pdl_trigger() (or has exited), i.e. while that kernel's last wave is
// still running; pdl_wait() then blocks until the kernel in front has COMPLETED and its writes are visible.  Rule kept
// everywhere: a kernel is launched through launch_pdl only if it calls pdl_wait() before its first access to global memory
// that any earlier kernel writes or still reads (tables written once at mk_create may be read earlier); kernels launched
// with <<< >>> keep the full serialisation.  MK_OPT_TUNE bit 12 launches everything without the attribute.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(const mk_ctx* c, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = c->stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = (c->tune & 4096) ? 0 : 1;
  return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}
#endif

// a block of consecutive receiver rows of R^ as one launch sees it: Rhat points at row r0 (its [nrow][nb][ld] block may be
// the resident part, a streaming window, or the mapped host part during ingest); S^ is indexed by the global receiver
struct RowBlock {
  float2* Rhat;
  int r0, nrow;
  int ld = 0;  // ingest only: elements between consecutive (receiver, bin) rows of the target (0 = the context's ld)
  int src_n = 0;  // ingest only: receivers per shot in the SOURCE array (0 = the context's nrec; mk_load_R_rows: its own rows)
};

// where a forward transform stores N^ (a1, a6)
constexpr int kMaxPeers = 7;  // other ranks of a row-sharded run whose operand receives this rank's rows directly

struct OperandOut {
  float2* plain;
  int ldf;
  // row of N^ that the trace of receiver r feeds: shot_of_rec[r] (-1: no source there, nothing is stored), nullptr = r
  const int* shot_of_rec;
  // row sharding with attached peers (mk_operand_attach): every store of this rank's rows goes to the same offset of
  // each peer's operand as well — the all-gather fused into the producing kernel as peer stores over NVLink
  int npeer;
  float2* peer[kMaxPeers];
};

int set_err(mk_ctx* c, int code, const std::string& msg);
int check_cuda(mk_ctx* c, cudaError_t e, const char* what);

// mk_fft_kernels.cu
int launch_window(mk_ctx* c, const float* d_td, int* d_h, int ntr);
int launch_load_R(mk_ctx* c, const RowBlock& rb, const float* d_R_time, int shot0, int nshots);
// time [nfoc][n][nt] -> Nhat band;  conj_out: spectrum of T(src);  d_init_Tsrc: optional, receives T src
int launch_fwd(mk_ctx* c, const float* d_src, const OperandOut& O, int nfoc, bool conj_out, float* d_init_Tsrc);
// spectrum [n][nb][ldf] -> out[j] = sS*S[j] + sA*A[j] + sB*B[(nt-j)%nt]
int launch_inv(mk_ctx* c, const float2* d_spec, int nfoc, int ldf, float* d_out, float sS, const float* d_A, float sA,
               const float* d_B, float sB);
// fused a3..a6
int launch_post(mk_ctx* c, const OperandOut& O, int parity_even, float* d_Ni_out);

// mk_syn_gemv.cu / mk_syn_gemm.cu:  Shat = Rhat x Nhat per bin
bool gemv_supported(const mk_ctx* c, int nfoc);
int launch_syn_gemv(mk_ctx* c, const RowBlock& rb, const float2* d_Nhat, float2* d_Shat, int nfoc);
int launch_syn_gemm(mk_ctx* c, const RowBlock& rb, const float2* d_Nhat, float2* d_Shat, int ldf);
// mk_syn_gemv_q16.cu: the streaming GEMV on block-float R^, and the quantiser of the ingest
int launch_syn_gemv_q16(mk_ctx* c, const float2* d_Nhat, float2* d_Shat, int nfoc);
int launch_quantize_q16(mk_ctx* c, const float2* d_stage, int ldc, int shot0);
// mk_syn_tc.cu: tcgen05 3xTF32 path.  slot: 0 = the run's operand, 1 = the scratch operand (descriptor cache)
bool tc_supported(const mk_ctx* c);
int launch_syn_tc(mk_ctx* c, const RowBlock& rb, int slot, const float2* d_Nhat, float2* d_Shat, int ldf);

}  // namespace mk

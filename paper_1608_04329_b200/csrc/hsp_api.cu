// hsp_api.cu -- the C-ABI boundary (include/hsp.h) and the host orchestrator of the sweep.
//
// Sweep DAG:   {a1 a2 a3 -> b}  ||  {e1 e2 -> c -> d1}  ->  d2 -> e3, g
// The Cholesky branch depends only on the previous beta, so it runs on a second stream beside the
// fused pass; one sweep is captured into a CUDA graph and replayed n_iter times (all kernel
// arguments that change between sweeps live in the device control block Ctl).
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <string>
#include <vector>
#include <algorithm>
#include <new>
#include <mutex>
#include "../../include/hsp.h"
#include "hsp_device.cuh"
#include "hsp_internal.h"

using namespace hsp;

static thread_local std::string g_err;
// process-wide defaults of the plan-time options (hsp_set_option with state == NULL); a chain copies them at create
static std::mutex g_opt_mutex;
static Options g_default_options;
static int fail(int code, const std::string& msg) { g_err = msg; return code; }
static int cuda_fail(cudaError_t e, const char* what) {
  g_err = std::string(what) + ": " + cudaGetErrorString(e);
  return e == cudaErrorMemoryAllocation ? HSP_ENOMEM : HSP_ECUDA;
}
#define CK(call)                                   \
  do {                                             \
    cudaError_t e_ = (call);                       \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call); \
  } while (0)

struct hsp_state {
  const void* X = nullptr; int dtype = 0; const unsigned char* y = nullptr; long long N = 0; int p = 0;
  long long row_offset = 0;          // global index of local row 0 (hsp_create_shard)
  unsigned long long seed = 0; cudaStream_t stream = nullptr; cudaStream_t stream2 = nullptr;
  cudaStream_t own_stream = nullptr;
  unsigned flags = 0; int num_sms = 0;
  void* own_X = nullptr; unsigned char* own_y = nullptr;
  const void* host_X = nullptr;      // hsp_create_host: X is uploaded in row chunks, overlapped with the Gram
  double *G = nullptr, *L = nullptr, *Lt = nullptr, *rv = nullptr, *W = nullptr, *Wt = nullptr, *beta = nullptr, *lam_inv2 = nullptr,
         *nu_inv = nullptr, *g = nullptr, *tv = nullptr, *partial = nullptr, *z = nullptr, *mu = nullptr;
  int pd_ctas = 0;                   // CTAs (= partial rows) of the paper-design X^T z product
  CholPlan chol{};
  signed char* side = nullptr;
  Ctl* ctl = nullptr;
  double *h_beta = nullptr, *h_lambda = nullptr, *h_tau = nullptr;
  long long h_cap = 0, h_n = 0, host_sweep = 0;
  bool z_valid = false;
  bool gram_tc = false;              // the Gram was computed on the tensor cores (gram_tc.cu)
  long long split_left = 0; bool split_open = false;   // hsp_sweep_prepare / _begin / _end
  int* h_status = nullptr;           // pinned host word for the status read of hsp_get_draws
  FusedPlan plan{};
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  cudaGraphExec_t graph_exec = nullptr; unsigned graph_flags = ~0u; long long graph_kernels = 0;
  long long launches = 0;
  std::vector<cudaEvent_t> tev;   // event pairs around the fused pass (direct-launch mode)
  size_t tev_used = 0; double fused_ms_sum = 0.0; long long fused_n = 0;
  Options opt{};                  // plan-time options, copied from the process defaults at create
  // asynchronous download of the draws (hsp_set_output): host ring + copy stream
  double *o_beta = nullptr, *o_lambda = nullptr, *o_tau = nullptr;   // HOST, borrowed
  long long o_cap = 0, o_rows = 0;         // ring capacity in sweeps; rows enqueued since hsp_set_output
  long long o_block = 1;                   // sweeps per download block
  long long o_pending_first = 0, o_pending = 0;   // history rows of the current call not yet handed to the copy stream
  cudaStream_t stream3 = nullptr;          // copy stream
  std::vector<cudaEvent_t> o_ev_sweep;     // recorded on the compute stream after the last sweep of a block
  std::vector<cudaEvent_t> o_ev_done;      // recorded on the copy stream after the block has landed on the host
  std::vector<long long> o_ev_rows;        // o_rows once that block is complete
  size_t o_ev_next = 0, o_ev_checked = 0; long long o_completed = 0;   // blocks enqueued / known landed; rows landed
  cudaEvent_t o_last_done = nullptr;       // the most recent o_ev_done (not owned)
};

static int prepare_history(hsp_state* s, long long n_iter);

static void free_state(hsp_state* s) {
  if (!s) return;
  if (s->graph_exec) cudaGraphExecDestroy(s->graph_exec);
  for (cudaEvent_t e : s->tev) cudaEventDestroy(e);
  if (s->ev_fork) cudaEventDestroy(s->ev_fork);
  if (s->ev_join) cudaEventDestroy(s->ev_join);
  for (cudaEvent_t e : s->o_ev_sweep) cudaEventDestroy(e);
  for (cudaEvent_t e : s->o_ev_done) cudaEventDestroy(e);
  if (s->stream3) cudaStreamDestroy(s->stream3);
  if (s->stream2) cudaStreamDestroy(s->stream2);
  if (s->own_stream) cudaStreamDestroy(s->own_stream);
  void* ptrs[] = {s->own_X, s->own_y, s->G, s->L, s->Lt, s->rv, s->W, s->Wt, s->beta, s->lam_inv2, s->nu_inv, s->g, s->tv, s->partial,
                  s->z, s->mu, s->side, s->ctl, s->h_beta, s->h_lambda, s->h_tau};
  for (void* q : ptrs) if (q) cudaFree(q);
  chol_plan_destroy(&s->chol);
  if (s->h_status) cudaFreeHost(s->h_status);
  delete s;
}

static int drain_fused_events(hsp_state* s) {
  for (size_t i = 0; i + 1 < s->tev_used; i += 2) {
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, s->tev[i], s->tev[i + 1]));
    s->fused_ms_sum += ms; s->fused_n += 1;
  }
  s->tev_used = 0;
  return HSP_OK;
}

// Enqueue one sweep.  `timed`: bracket the fused pass with CUDA events (direct-launch mode only).
//   stream A:  fused pass (a1-a3) ------------------------------> [join] reduce (b) -> d2 (two products; k <- k+1)
//   stream B:  scales (e1, e2, e3; lambda, tau history) -> Q build + Cholesky + inverse factor (c, d1)
// phases: 1 = up to and including the reduction of X^T z (and the whole side branch), 2 = the beta draw, 3 = both.
static int enqueue_sweep(hsp_state* s, bool timed, long long* kernels, int phases = 3) {
  cudaStream_t A = s->stream;
  // one stream when asked for, and when the plan found no way to hide the Cholesky branch (c, d1) behind the pass
  // (p = 4000: both kernels want every SM; launched on two streams their CTAs would interleave at random)
  const bool serial = (s->flags & HSP_SERIAL) != 0 || !s->chol.overlap;
  cudaStream_t B = serial ? A : s->stream2;
  const bool do_z = !(s->flags & HSP_FREEZE_Z), do_scales = !(s->flags & HSP_FREEZE_SCALES),
             do_beta = !(s->flags & HSP_FREEZE_BETA);
  if (phases == 2) goto draw;
  if (!serial) {
    CK(cudaEventRecord(s->ev_fork, A));
    CK(cudaStreamWaitEvent(B, s->ev_fork, 0));
  }
  {
  auto side_branch = [&]() -> int {
    CK(scales_launch(s->beta, s->lam_inv2, s->nu_inv, s->ctl, s->p, s->seed, do_scales ? 0 : 1, B));
    *kernels += 1;
    if (do_beta) CK(cholesky_launch(s->chol, s->G, s->lam_inv2, s->ctl, s->L, s->W, s->Wt, s->Lt, B, kernels));
    return HSP_OK;
  };
  if (serial) { const int rc = side_branch(); if (rc) return rc; }
  if (do_z) {
    if (timed) {
      if (s->tev_used + 2 > s->tev.size()) {
        for (int q = 0; q < 2; ++q) { cudaEvent_t e; CK(cudaEventCreate(&e)); s->tev.push_back(e); }
      }
      CK(cudaEventRecord(s->tev[s->tev_used], A));
    }
    if (s->flags & HSP_PAPER_DESIGN) {
      CK(paper_design_launch(s->X, s->dtype, s->y, s->N, s->p, s->seed, s->beta, s->ctl, s->mu, s->z, s->partial,
                             s->pd_ctas, s->num_sms, A));
      *kernels += 2;
    } else {
      CK(fused_pass_launch(s->plan, s->X, s->dtype, s->y, s->N, s->p, s->seed, s->beta, s->ctl, s->partial,
                           (s->flags & HSP_STORE_Z) ? s->z : nullptr, A));
    }
    if (timed) { CK(cudaEventRecord(s->tev[s->tev_used + 1], A)); s->tev_used += 2; }
    *kernels += 1;
  }
  if (!serial) {
    const int rc = side_branch(); if (rc) return rc;
    CK(cudaEventRecord(s->ev_join, B));
    CK(cudaStreamWaitEvent(A, s->ev_join, 0));      // before the reduce: the tail kernels then chain by PDL
  }
  if (do_z) {
    const int n_part = (s->flags & HSP_PAPER_DESIGN) ? s->pd_ctas : s->plan.grid * s->plan.groups;
    CK(reduce_partials_launch(s->partial, n_part, s->p, s->g, A));
    *kernels += 1;
  }
  }
  if (phases == 1) return HSP_OK;
draw:
  if (do_beta && s->chol.sb < s->chol.nt)
    CK(beta_block_solve_launch(s->L, s->Lt, s->W, s->Wt, s->g, s->tv, s->rv, s->beta, s->p, s->chol.sb, s->seed, s->ctl, A, kernels,
                               opt_or(s->opt.no_pdl, 0) == 0));
  else if (do_beta) CK(beta_solve_launch(s->W, s->Wt, s->g, s->tv, s->beta, s->p, s->seed, s->ctl, A, kernels, opt_or(s->opt.no_pdl, 0) == 0));
  else { CK(beta_keep_launch(s->beta, s->p, s->ctl, A)); *kernels += 1; }
  return HSP_OK;
}

static int build_graph(hsp_state* s) {
  if (s->graph_exec) { cudaGraphExecDestroy(s->graph_exec); s->graph_exec = nullptr; }
  cudaGraph_t graph = nullptr;
  CK(cudaStreamBeginCapture(s->stream, cudaStreamCaptureModeThreadLocal));
  long long kernels = 0;
  const int rc = enqueue_sweep(s, false, &kernels);
  cudaError_t e = cudaStreamEndCapture(s->stream, &graph);
  if (rc != HSP_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
  if (e != cudaSuccess) return cuda_fail(e, "cudaStreamEndCapture");
  e = cudaGraphInstantiate(&s->graph_exec, graph, 0);
  cudaGraphDestroy(graph);
  if (e != cudaSuccess) return cuda_fail(e, "cudaGraphInstantiate");
  s->graph_flags = s->flags; s->graph_kernels = kernels;
  return HSP_OK;
}

static int create_common(hsp_state** out, hsp_state* s) {
  const int p = s->p; const long long N = s->N;
  int dev = 0;
  CK(cudaGetDevice(&dev));
  if (s->stream == nullptr) {
    // the legacy default stream cannot be captured into a graph: use a blocking stream of our own,
    // which still orders itself after/before work on the legacy stream
    CK(cudaStreamCreateWithFlags(&s->own_stream, cudaStreamDefault));
    s->stream = s->own_stream;
  }
  CK(cudaDeviceGetAttribute(&s->num_sms, cudaDevAttrMultiProcessorCount, dev));
  CK(cudaStreamCreateWithFlags(&s->stream2, cudaStreamNonBlocking));
  CK(cudaEventCreateWithFlags(&s->ev_fork, cudaEventDisableTiming));
  CK(cudaEventCreateWithFlags(&s->ev_join, cudaEventDisableTiming));
  // SM budget: when the Cholesky branch (c, d1) can hide behind the fused pass it gets chol_ctas SMs of
  // its own and the pass the rest; otherwise both use every SM and run one after the other.
  const double x_bytes = (double)N * p * (s->dtype == HSP_F32 ? 4.0 : 8.0);
  const double fused_ms_est = x_bytes / 7.0e9 + 0.01;   // the pass streams X at ~7.2 TB/s on B200 (profiles/)
  { std::lock_guard<std::mutex> lock(g_opt_mutex); s->opt = g_default_options; }
  CK(chol_plan_create(&s->chol, p, s->num_sms, fused_ms_est, s->opt));
  // Two SMs are left to neither: with every SM spoken for, a single SM that is busy for a moment when the Cholesky branch
  // starts (any other kernel of the process, a driver-side copy kernel) leaves one of its CTAs without a home until the
  // persistent pass ends -- and the tiles that CTA owns stall the whole task graph: the sweep then takes pass + branch
  // instead of max(pass, branch).  Measured by forcing one CTA too many: C3 0.583 -> 0.878 ms, C4 1.52 -> 2.73 ms; the same
  // signature showed up unforced in about one bench run in ten.  The pass is HBM-bound with SMs to spare (8.1): 130 instead
  // of 132 CTAs cost < 1 %.
  const int kSpareSms = 2;
  const int fused_sms = s->chol.overlap ? std::max(1, s->num_sms - s->chol.K - kSpareSms) : s->num_sms;
  s->plan = fused_plan(s->dtype, N, p, fused_sms, s->X, s->opt);
  s->plan.row_offset = s->row_offset;
  // set opt-in shared-memory attributes now, outside any stream capture
  CK(fused_pass_launch(s->plan, s->X, s->dtype, s->y, -1, p, 0, nullptr, nullptr, nullptr, nullptr, s->stream));
  const size_t pp = (size_t)p * p * sizeof(double), pv = (size_t)p * sizeof(double);
  const size_t P = (size_t)chol_ld(p), PP = P * P * sizeof(double), Pv = P * sizeof(double);
  CK(cudaMalloc(&s->G, pp)); CK(cudaMalloc(&s->L, PP)); CK(cudaMalloc(&s->W, PP)); CK(cudaMalloc(&s->Wt, PP));
  CK(cudaMalloc(&s->beta, Pv));   // beta padded to P with zeros (the block solve reads whole tiles)
  CK(cudaMalloc(&s->lam_inv2, pv)); CK(cudaMalloc(&s->nu_inv, pv));
  CK(cudaMalloc(&s->g, Pv)); CK(cudaMalloc(&s->tv, Pv));     // padded to P with zeros (the GEMVs read whole tiles)
  s->pd_ctas = paper_design_ctas(N, s->num_sms);
  CK(cudaMalloc(&s->partial, (size_t)std::max(s->plan.grid * s->plan.groups, s->pd_ctas) * pv));
  CK(cudaMalloc(&s->ctl, sizeof(Ctl)));
  CK(cudaMallocHost(&s->h_status, sizeof(int)));
  // validate y in {0,1}
  int* bad = nullptr;
  CK(cudaMalloc(&bad, sizeof(int)));
  CK(cudaMemsetAsync(bad, 0, sizeof(int), s->stream));
  CK(validate_y_launch(s->y, N, bad, s->stream));
  int h_bad = 0;
  CK(cudaMemcpyAsync(&h_bad, bad, sizeof(int), cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  cudaFree(bad);
  s->launches += 1;
  if (h_bad) return fail(HSP_EINVAL, "y must contain only 0 and 1");
  // cold start: beta = 0; lambda = nu = tau = xi = 1
  std::vector<double> ones((size_t)p, 1.0);
  CK(cudaMemsetAsync(s->beta, 0, Pv, s->stream));
  if (s->chol.sb < s->chol.nt) {
    CK(cudaMalloc(&s->Lt, PP)); CK(cudaMalloc(&s->rv, Pv));
    CK(cudaMemsetAsync(s->Lt, 0, PP, s->stream)); CK(cudaMemsetAsync(s->rv, 0, Pv, s->stream));
    CK(cudaMemsetAsync(s->W, 0, PP, s->stream)); CK(cudaMemsetAsync(s->Wt, 0, PP, s->stream));
  }
  CK(cudaMemsetAsync(s->g, 0, Pv, s->stream));
  CK(cudaMemsetAsync(s->tv, 0, Pv, s->stream));
  CK(cudaMemsetAsync(s->L, 0, PP, s->stream));
  CK(cudaMemcpyAsync(s->lam_inv2, ones.data(), pv, cudaMemcpyHostToDevice, s->stream));
  CK(cudaMemcpyAsync(s->nu_inv, ones.data(), pv, cudaMemcpyHostToDevice, s->stream));
  Ctl c{}; c.sweep = 0; c.hist_base = 0; c.tau_inv2 = 1.0; c.xi_inv = 1.0; c.status = 0; c.done = 0;
  c.h_beta = c.h_lambda = c.h_tau = nullptr;
  CK(cudaMemcpyAsync(s->ctl, &c, sizeof(Ctl), cudaMemcpyHostToDevice, s->stream));
  CK(cudaStreamSynchronize(s->stream));   // `ones` and `c` are stack/heap temporaries
  // c0: G = X^T X once, by row chunks; with host input the upload of chunk c+1 (copy stream) runs
  // beside the Gram of chunk c
  // fp32 X and a large contraction: tcgen05 tensor cores (split-bf16 products, fp64 flush; ~1e-7 relative);
  // otherwise exact fp64 DFMA tiles.  Option "gram_tc" = 0 / 1 forces the choice.
  const bool use_tc = s->dtype == HSP_F32 && (s->opt.gram_tc >= 0 ? s->opt.gram_tc != 0 : (double)N * p * p >= 2e10);
  s->gram_tc = use_tc;
  const GramPlan gp = gram_plan(N, p, s->dtype, s->num_sms, use_tc);
  double* scratch = s->W;                  // W (>= p*p doubles) is free until the first sweep
  if (gp.slots > 1) CK(cudaMalloc(&scratch, (size_t)gp.slots * pp));
  cudaError_t e = cudaSuccess;
  const size_t row_bytes = (size_t)p * (s->dtype == HSP_F32 ? 4 : 8);
  const long long chunk_rows = gp.rows_per_slot * gp.slots_per_chunk;
  for (int c = 0; c < gp.chunks && e == cudaSuccess; ++c) {
    if (s->host_X != nullptr) {
      const long long r0 = (long long)c * chunk_rows;
      const long long r1 = (c == gp.chunks - 1) ? N : std::min(N, r0 + chunk_rows);
      if (r1 > r0) {
        e = cudaMemcpyAsync(static_cast<char*>(s->own_X) + (size_t)r0 * row_bytes,
                            static_cast<const char*>(s->host_X) + (size_t)r0 * row_bytes, (size_t)(r1 - r0) * row_bytes,
                            cudaMemcpyHostToDevice, s->stream2);
        if (e == cudaSuccess) e = cudaEventRecord(s->ev_fork, s->stream2);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(s->stream, s->ev_fork, 0);
      }
    }
    if (e == cudaSuccess)
      e = use_tc ? gram_tc_chunk_launch(gp, c, static_cast<const float*>(s->X), N, p, scratch, s->stream)
                 : gram_chunk_launch(gp, c, s->X, s->dtype, N, p, scratch, s->stream);
  }
  if (e == cudaSuccess) e = gram_finish_launch(gp, p, scratch, s->G, s->stream);
  s->launches += gp.chunks + 2;
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  if (gp.slots > 1) cudaFree(scratch);
  if (e != cudaSuccess) return cuda_fail(e, "gram");
  *out = s;
  return HSP_OK;
}

// ---- asynchronous download of the draws (hsp_set_output; "Monte Carlo output is downloaded off of the
// GPU at the same time as updates for other variables are computed").  The device history of the current call holds
// rows [0, h_n); after the last sweep of a block of o_block sweeps has been enqueued, an event is recorded on the compute
// stream, the copy stream waits for it and copies the block's rows of beta, lambda, tau into the host ring, and a second
// event marks the block as landed.  Nothing here synchronises the host.
static const size_t kOutEvents = 4096;   // event pairs kept before the oldest is waited for and reused

static int output_flush(hsp_state* s) {
  if (s->o_cap <= 0 || s->o_pending <= 0) { s->o_pending = 0; return HSP_OK; }
  const size_t slot = s->o_ev_next % kOutEvents;
  if (s->o_ev_sweep.size() <= slot) {
    cudaEvent_t a, b;
    CK(cudaEventCreateWithFlags(&a, cudaEventDisableTiming));
    CK(cudaEventCreateWithFlags(&b, cudaEventDisableTiming));
    s->o_ev_sweep.push_back(a); s->o_ev_done.push_back(b); s->o_ev_rows.push_back(0);
  } else {
    CK(cudaEventSynchronize(s->o_ev_done[slot]));     // kOutEvents blocks ago; makes the event pair reusable
    s->o_completed = std::max(s->o_completed, s->o_ev_rows[slot]);
    s->o_ev_checked = std::max(s->o_ev_checked, s->o_ev_next + 1 - kOutEvents);
  }
  CK(cudaEventRecord(s->o_ev_sweep[slot], s->stream));
  CK(cudaStreamWaitEvent(s->stream3, s->o_ev_sweep[slot], 0));
  const int p = s->p;
  long long src = s->o_pending_first, left = s->o_pending;
  while (left > 0) {
    const long long dst = s->o_rows % s->o_cap;
    const long long n = std::min(left, s->o_cap - dst);
    if (s->o_beta) CK(cudaMemcpyAsync(s->o_beta + (size_t)dst * p, s->h_beta + (size_t)src * p, (size_t)n * p * sizeof(double), cudaMemcpyDeviceToHost, s->stream3));
    if (s->o_lambda) CK(cudaMemcpyAsync(s->o_lambda + (size_t)dst * p, s->h_lambda + (size_t)src * p, (size_t)n * p * sizeof(double), cudaMemcpyDeviceToHost, s->stream3));
    if (s->o_tau) CK(cudaMemcpyAsync(s->o_tau + dst, s->h_tau + src, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, s->stream3));
    s->o_rows += n; src += n; left -= n;
  }
  CK(cudaMemcpyAsync(s->h_status, reinterpret_cast<const char*>(s->ctl) + offsetof(Ctl, status), sizeof(int), cudaMemcpyDeviceToHost, s->stream3));
  CK(cudaEventRecord(s->o_ev_done[slot], s->stream3));
  s->o_ev_rows[slot] = s->o_rows;
  s->o_last_done = s->o_ev_done[slot];
  s->o_ev_next += 1;
  s->o_pending_first += s->o_pending; s->o_pending = 0;
  return HSP_OK;
}

// one more sweep of the current call has been enqueued on the compute stream
static int output_after_sweep(hsp_state* s, bool last_of_call) {
  if (s->o_cap <= 0) return HSP_OK;
  s->o_pending += 1;
  if (s->o_pending >= s->o_block || last_of_call) return output_flush(s);
  return HSP_OK;
}

// Device history for at least n_iter sweeps.  Growing it synchronises the chain and calls cudaFree / cudaMalloc, which on
// the boxes this was measured on occasionally takes 0.1 - 1 s (seen as a few per cent of hsp_sweep calls that "took twice as
// long": the GPU sits idle meanwhile): callers that time sweeps reserve the capacity first (hsp_reserve_history).
static int grow_history(hsp_state* s, long long n_iter) {
  if (n_iter <= s->h_cap) return HSP_OK;
  const int p = s->p;
  CK(cudaStreamSynchronize(s->stream));
  if (s->stream3) CK(cudaStreamSynchronize(s->stream3));
  if (s->h_beta) { cudaFree(s->h_beta); cudaFree(s->h_lambda); cudaFree(s->h_tau); s->h_beta = s->h_lambda = s->h_tau = nullptr; }
  s->h_cap = 0; s->h_n = 0;
  CK(cudaMalloc(&s->h_beta, (size_t)n_iter * p * sizeof(double)));
  CK(cudaMalloc(&s->h_lambda, (size_t)n_iter * p * sizeof(double)));
  CK(cudaMalloc(&s->h_tau, (size_t)n_iter * sizeof(double)));
  s->h_cap = n_iter;
  return HSP_OK;
}

static int prepare_history(hsp_state* s, long long n_iter) {
  // the copy stream may still be reading the history of the previous call: the new call's sweeps start after it
  if (s->o_last_done) CK(cudaStreamWaitEvent(s->stream, s->o_last_done, 0));
  s->o_pending_first = 0; s->o_pending = 0;
  { const int rc = grow_history(s, n_iter); if (rc != HSP_OK) return rc; }
  s->h_n = n_iter;
  if (n_iter == 0) return HSP_OK;
  // history window of this call: set by a one-thread kernel (its arguments are copied at launch: no host sync)
  CK(set_history_launch(s->ctl, (unsigned long long)s->host_sweep, s->h_beta, s->h_lambda, s->h_tau, s->stream));
  s->launches += 1;
  return HSP_OK;
}

static int create_device(hsp_state** out, const void* X, int x_dtype, const unsigned char* y, long long N, int p,
                         unsigned long long seed, long long row_offset, void* stream) {
  if (!out) return fail(HSP_EINVAL, "out is NULL");
  *out = nullptr;
  if (!X || !y) return fail(HSP_EINVAL, "X or y is NULL");
  if (x_dtype != HSP_F32 && x_dtype != HSP_F64) return fail(HSP_EINVAL, "x_dtype must be HSP_F32 or HSP_F64");
  if (N < 2) return fail(HSP_EINVAL, "N must be >= 2");
  if (p < 1) return fail(HSP_EINVAL, "p must be >= 1");
  if (row_offset < 0) return fail(HSP_EINVAL, "row_offset must be >= 0");
  if (reinterpret_cast<uintptr_t>(X) % (x_dtype == HSP_F32 ? 4 : 8)) return fail(HSP_EINVAL, "X is misaligned");
  cudaPointerAttributes pa{};
  if (cudaPointerGetAttributes(&pa, X) != cudaSuccess || (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged)) {
    cudaGetLastError();
    return fail(HSP_EINVAL, "X must be a device pointer");
  }
  if (cudaPointerGetAttributes(&pa, y) != cudaSuccess || (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged)) {
    cudaGetLastError();
    return fail(HSP_EINVAL, "y must be a device pointer");
  }
  hsp_state* s = new (std::nothrow) hsp_state();
  if (!s) return fail(HSP_ENOMEM, "out of host memory");
  s->X = X; s->dtype = x_dtype; s->y = y; s->N = N; s->p = p; s->seed = seed; s->stream = (cudaStream_t)stream;
  s->row_offset = row_offset;
  const int rc = create_common(out, s);
  if (rc != HSP_OK) { free_state(s); *out = nullptr; }
  return rc;
}

extern "C" {

const char* hsp_last_error(void) { return g_err.c_str(); }

int hsp_create(hsp_state** out, const void* X, int x_dtype, const unsigned char* y, long long N, int p,
               unsigned long long seed, void* stream) {
  return create_device(out, X, x_dtype, y, N, p, seed, 0, stream);
}

int hsp_create_host(hsp_state** out, const void* X_host, int x_dtype, const unsigned char* y_host, long long N, int p,
                    unsigned long long seed, void* stream) {
  if (!out) return fail(HSP_EINVAL, "out is NULL");
  *out = nullptr;
  if (!X_host || !y_host) return fail(HSP_EINVAL, "X or y is NULL");
  if (x_dtype != HSP_F32 && x_dtype != HSP_F64) return fail(HSP_EINVAL, "x_dtype must be HSP_F32 or HSP_F64");
  if (N < 2) return fail(HSP_EINVAL, "N must be >= 2");
  if (p < 1) return fail(HSP_EINVAL, "p must be >= 1");
  hsp_state* s = new (std::nothrow) hsp_state();
  if (!s) return fail(HSP_ENOMEM, "out of host memory");
  s->dtype = x_dtype; s->N = N; s->p = p; s->seed = seed; s->stream = (cudaStream_t)stream;
  const size_t xb = (size_t)N * p * (x_dtype == HSP_F32 ? 4 : 8);
  cudaError_t e = cudaMalloc(&s->own_X, xb);
  if (e == cudaSuccess) e = cudaMalloc(&s->own_y, (size_t)N);
  if (e == cudaSuccess) e = cudaMemcpyAsync(s->own_y, y_host, (size_t)N, cudaMemcpyHostToDevice, s->stream);
  if (e != cudaSuccess) { const int rc = cuda_fail(e, "allocation / upload of y"); free_state(s); return rc; }
  s->X = s->own_X; s->y = s->own_y; s->host_X = X_host;   // X itself is uploaded chunk by chunk in create_common
  const int rc = create_common(out, s);
  if (rc != HSP_OK) { free_state(s); *out = nullptr; }
  return rc;
}

int hsp_create_shard(hsp_state** out, const void* X, int x_dtype, const unsigned char* y, long long N_local, int p,
                     unsigned long long seed, long long row_offset, void* stream) {
  return create_device(out, X, x_dtype, y, N_local, p, seed, row_offset, stream);
}

int hsp_sweep_prepare(hsp_state* s, long long n_iter) {
  if (!s) return fail(HSP_EINVAL, "state is NULL");
  if (n_iter < 0) return fail(HSP_EINVAL, "n_iter must be >= 0");
  if (s->flags & HSP_PAPER_DESIGN) return fail(HSP_EINVAL, "HSP_PAPER_DESIGN is not available for sharded sweeps");
  s->split_left = n_iter; s->split_open = false;
  return prepare_history(s, n_iter);
}

int hsp_sweep_begin(hsp_state* s) {
  if (!s) return fail(HSP_EINVAL, "state is NULL");
  if (s->split_left <= 0 || s->split_open) return fail(HSP_EINVAL, "hsp_sweep_begin: call hsp_sweep_prepare first / finish the open sweep");
  if (s->flags & HSP_STORE_Z) s->z_valid = !(s->flags & HSP_FREEZE_Z) || s->z_valid;
  else if (!(s->flags & HSP_FREEZE_Z)) s->z_valid = false;
  if (s->tev_used >= 8192) { CK(cudaStreamSynchronize(s->stream)); const int rc = drain_fused_events(s); if (rc) return rc; }
  long long k = 0;
  const int rc = enqueue_sweep(s, (s->flags & HSP_NO_GRAPH) != 0, &k, 1);
  if (rc != HSP_OK) return rc;
  s->launches += k; s->split_open = true;
  return HSP_OK;
}

int hsp_sweep_end(hsp_state* s) {
  if (!s) return fail(HSP_EINVAL, "state is NULL");
  if (!s->split_open) return fail(HSP_EINVAL, "hsp_sweep_end without hsp_sweep_begin");
  long long k = 0;
  const int rc = enqueue_sweep(s, false, &k, 2);
  if (rc != HSP_OK) return rc;
  s->launches += k; s->split_open = false; s->split_left -= 1; s->host_sweep += 1;
  return output_after_sweep(s, s->split_left == 0);
}

double* hsp_xtz_device(hsp_state* s) { return s ? s->g : nullptr; }
double* hsp_gram_device(hsp_state* s) { return s ? s->G : nullptr; }

int hsp_destroy(hsp_state* s) {
  if (!s) return HSP_OK;
  cudaStreamSynchronize(s->stream);
  if (s->stream2) cudaStreamSynchronize(s->stream2);
  if (s->stream3) cudaStreamSynchronize(s->stream3);
  free_state(s);
  return HSP_OK;
}

static int* option_slot(Options& o, const char* key) {
  struct { const char* name; int Options::*field; } const table[] = {
      {"fused_eta", &Options::fused_eta}, {"fused_grid", &Options::fused_grid}, {"fused_stages", &Options::fused_stages},
      {"fused_lag", &Options::fused_lag}, {"fused_w", &Options::fused_w}, {"narrow_rt", &Options::narrow_rt},
      {"fused_variant", &Options::fused_variant}, {"fused_narrow", &Options::fused_narrow}, {"chol_ctas", &Options::chol_ctas},
      {"chol_sb", &Options::chol_sb}, {"chol_trace", &Options::chol_trace}, {"gram_tc", &Options::gram_tc},
      {"no_pdl", &Options::no_pdl}};
  for (const auto& t : table)
    if (strcmp(t.name, key) == 0) return &(o.*(t.field));
  return nullptr;
}

int hsp_set_option(hsp_state* s, const char* key, long long value) {
  if (value > 0x7fffffffLL) return fail(HSP_EINVAL, "option value out of range");
  const int v = value < 0 ? -1 : (int)value;
  if (s == nullptr) {
    std::lock_guard<std::mutex> lock(g_opt_mutex);
    if (key == nullptr) { g_default_options = Options{}; return HSP_OK; }
    int* slot = option_slot(g_default_options, key);
    if (!slot) return fail(HSP_EINVAL, std::string("unknown option: ") + key);
    *slot = v;
    return HSP_OK;
  }
  // an existing chain: its launch plan is fixed; only the launch-mode option can change
  if (key == nullptr) return fail(HSP_EINVAL, "key is NULL");
  if (strcmp(key, "no_pdl") != 0) {
    Options probe;
    if (!option_slot(probe, key)) return fail(HSP_EINVAL, std::string("unknown option: ") + key);
    return fail(HSP_EINVAL, std::string("plan-time option (set it with state = NULL before hsp_create): ") + key);
  }
  s->opt.no_pdl = v;
  s->graph_flags = ~0u;        // the captured graph is rebuilt by the next hsp_sweep
  return HSP_OK;
}

int hsp_get_option(const hsp_state* s, const char* key, long long* value) {
  if (!key || !value) return fail(HSP_EINVAL, "NULL argument");
  Options o;
  if (s) o = s->opt; else { std::lock_guard<std::mutex> lock(g_opt_mutex); o = g_default_options; }
  int* slot = option_slot(o, key);
  if (!slot) return fail(HSP_EINVAL, std::string("unknown option: ") + key);
  *value = *slot;
  return HSP_OK;
}

int hsp_set_output(hsp_state* s, double* host_beta, double* host_lambda, double* host_tau, long long capacity) {
  if (!s) return fail(HSP_EINVAL, "state is NULL");
  if (capacity < 0) return fail(HSP_EINVAL, "capacity must be >= 0");
  if (s->split_open) return fail(HSP_EINVAL, "hsp_set_output between hsp_sweep_begin and hsp_sweep_end");
  // blocks in flight target the old buffers: let them land first
  if (s->stream3) CK(cudaStreamSynchronize(s->stream3));
  if (capacity == 0 || (!host_beta && !host_lambda && !host_tau)) {
    s->o_beta = s->o_lambda = s->o_tau = nullptr; s->o_cap = 0; s->o_rows = 0; s->o_completed = 0; s->o_pending = 0;
    s->o_ev_checked = s->o_ev_next;
    return HSP_OK;
  }
  if (!s->stream3) CK(cudaStreamCreateWithFlags(&s->stream3, cudaStreamNonBlocking));
  s->o_beta = host_beta; s->o_lambda = host_lambda; s->o_tau = host_tau; s->o_cap = capacity;
  s->o_rows = 0; s->o_completed = 0; s->o_pending = 0;
  s->o_pending_first = s->h_n - s->split_left;        // only sweeps enqueued from now on
  s->o_ev_checked = s->o_ev_next;
  // sweeps per download block: at least ~64 KB per block, so that small problems are not bound by copy launches
  const long long row_bytes = (long long)(2 * s->p + 1) * (long long)sizeof(double);
  s->o_block = std::max<long long>(1, std::min<long long>((65536 + row_bytes - 1) / row_bytes, std::max<long long>(1, capacity / 2)));
  return HSP_OK;
}

int hsp_output_wait(hsp_state* s, long long* rows) {
  if (!s) return fail(HSP_EINVAL, "state is NULL");
  if (s->o_cap > 0 && s->o_pending > 0) { const int rc = output_flush(s); if (rc != HSP_OK) return rc; }
  if (s->o_last_done) CK(cudaEventSynchronize(s->o_last_done));
  s->o_completed = s->o_rows; s->o_ev_checked = s->o_ev_next;
  if (rows) *rows = s->o_rows;
  if (s->o_last_done) {
    if (*s->h_status == HSP_ENOTPD) return fail(HSP_ENOTPD, "Cholesky breakdown: Q is not positive definite");
    if (*s->h_status == HSP_ENUMERIC) return fail(HSP_ENUMERIC, "non-finite value in the chain state");
  }
  return HSP_OK;
}

int hsp_output_ready(hsp_state* s, long long* rows) {
  if (!s || !rows) return fail(HSP_EINVAL, "NULL argument");
  // non-blocking: advance over the blocks whose "landed" event has completed, oldest first
  while (s->o_ev_checked < s->o_ev_next) {
    const size_t slot = s->o_ev_checked % kOutEvents;
    const cudaError_t e = cudaEventQuery(s->o_ev_done[slot]);
    if (e == cudaErrorNotReady) break;
    if (e != cudaSuccess) return cuda_fail(e, "cudaEventQuery");
    s->o_completed = std::max(s->o_completed, s->o_ev_rows[slot]);
    s->o_ev_checked += 1;
  }
  *rows = s->o_completed;
  return HSP_OK;
}

int hsp_set_flags(hsp_state* s, unsigned flags) {
  if (!s) return fail(HSP_EINVAL, "state is NULL");
  const unsigned known = HSP_STORE_Z | HSP_FREEZE_SCALES | HSP_FREEZE_Z | HSP_FREEZE_BETA | HSP_NO_GRAPH | HSP_SERIAL |
                         HSP_PAPER_DESIGN;
  if (flags & ~known) return fail(HSP_EINVAL, "unknown flag");
  if (flags & HSP_PAPER_DESIGN) flags |= HSP_STORE_Z;   // the paper's design materialises z (and mu) in HBM
  if ((flags & HSP_PAPER_DESIGN) && !s->mu) CK(cudaMalloc(&s->mu, (size_t)s->N * sizeof(double)));
  if ((flags & HSP_STORE_Z) && !s->z) {
    CK(cudaMalloc(&s->z, (size_t)s->N * sizeof(double)));
    CK(cudaMemsetAsync(s->z, 0, (size_t)s->N * sizeof(double), s->stream));
  }
  s->flags = flags;
  return HSP_OK;
}

int hsp_reserve_history(hsp_state* s, long long n_iter) {
  if (!s) return fail(HSP_EINVAL, "state is NULL");
  if (n_iter < 0) return fail(HSP_EINVAL, "n_iter must be >= 0");
  if (s->split_open) return fail(HSP_EINVAL, "hsp_reserve_history between hsp_sweep_begin and hsp_sweep_end");
  if (s->split_left > 0 && n_iter > s->h_cap) return fail(HSP_EINVAL, "hsp_reserve_history inside a prepared run of sharded sweeps");
  return grow_history(s, n_iter);
}

int hsp_sweep(hsp_state* s, long long n_iter) {
  if (!s) return fail(HSP_EINVAL, "state is NULL");
  if (n_iter < 0) return fail(HSP_EINVAL, "n_iter must be >= 0");
  s->split_left = 0; s->split_open = false;
  { const int rc = prepare_history(s, n_iter); if (rc != HSP_OK) return rc; }
  if (n_iter == 0) return HSP_OK;
  if (s->flags & HSP_STORE_Z) s->z_valid = !(s->flags & HSP_FREEZE_Z) || s->z_valid;
  else if (!(s->flags & HSP_FREEZE_Z)) s->z_valid = false;
  if (s->flags & HSP_NO_GRAPH) {
    for (long long it = 0; it < n_iter; ++it) {
      if (s->tev_used >= 8192) { CK(cudaStreamSynchronize(s->stream)); const int rc = drain_fused_events(s); if (rc) return rc; }
      long long k = 0;
      const int rc = enqueue_sweep(s, true, &k);
      if (rc != HSP_OK) return rc;
      s->launches += k;
      const int rc2 = output_after_sweep(s, it == n_iter - 1); if (rc2 != HSP_OK) return rc2;
    }
  } else {
    if (!s->graph_exec || s->graph_flags != s->flags) {
      const int rc = build_graph(s);
      if (rc != HSP_OK) return rc;
    }
    for (long long it = 0; it < n_iter; ++it) {
      CK(cudaGraphLaunch(s->graph_exec, s->stream));
      const int rc2 = output_after_sweep(s, it == n_iter - 1); if (rc2 != HSP_OK) return rc2;
    }
    s->launches += s->graph_kernels * n_iter;
  }
  s->host_sweep += n_iter;
  return HSP_OK;
}

static int sync_status(const hsp_state* s) {
  CK(cudaStreamSynchronize(s->stream));
  int st = 0;
  CK(cudaMemcpy(&st, reinterpret_cast<const char*>(s->ctl) + offsetof(Ctl, status), sizeof(int), cudaMemcpyDeviceToHost));
  if (st == HSP_ENOTPD) return fail(HSP_ENOTPD, "Cholesky breakdown: Q is not positive definite");
  if (st == HSP_ENUMERIC) return fail(HSP_ENUMERIC, "non-finite value in the chain state");
  return HSP_OK;
}

int hsp_sync(const hsp_state* s) {
  if (!s) return fail(HSP_EINVAL, "state is NULL");
  return sync_status(s);
}

int hsp_get_draws(const hsp_state* s, double* beta, double* lambda, double* tau) {
  if (!s) return fail(HSP_EINVAL, "state is NULL");
  // status and draws are copied on the stream and the stream is synchronised once
  const size_t np = (size_t)s->h_n * s->p * sizeof(double);
  int* st = s->h_status;
  CK(cudaMemcpyAsync(st, reinterpret_cast<const char*>(s->ctl) + offsetof(Ctl, status), sizeof(int), cudaMemcpyDeviceToHost, s->stream));
  if (s->h_n > 0) {
    if (beta) CK(cudaMemcpyAsync(beta, s->h_beta, np, cudaMemcpyDefault, s->stream));
    if (lambda) CK(cudaMemcpyAsync(lambda, s->h_lambda, np, cudaMemcpyDefault, s->stream));
    if (tau) CK(cudaMemcpyAsync(tau, s->h_tau, (size_t)s->h_n * sizeof(double), cudaMemcpyDefault, s->stream));
  }
  CK(cudaStreamSynchronize(s->stream));
  if (*st == HSP_ENOTPD) return fail(HSP_ENOTPD, "Cholesky breakdown: Q is not positive definite");
  if (*st == HSP_ENUMERIC) return fail(HSP_ENUMERIC, "non-finite value in the chain state");
  return HSP_OK;
}

int hsp_get_latent(const hsp_state* s, double* z, signed char* side) {
  if (!s) return fail(HSP_EINVAL, "state is NULL");
  CK(cudaStreamSynchronize(s->stream));
  if (z) {
    if (!s->z || !s->z_valid) return fail(HSP_EINVAL, "z was not stored: set HSP_STORE_Z before hsp_sweep");
    CK(cudaMemcpy(z, s->z, (size_t)s->N * sizeof(double), cudaMemcpyDefault));
  }
  if (side) {
    hsp_state* m = const_cast<hsp_state*>(s);
    if (!m->side) CK(cudaMalloc(&m->side, (size_t)s->N));
    CK(side_launch(s->y, s->N, m->side, s->stream));
    m->launches += 1;
    CK(cudaStreamSynchronize(s->stream));
    CK(cudaMemcpy(side, m->side, (size_t)s->N, cudaMemcpyDefault));
  }
  return HSP_OK;
}

int hsp_get_state(const hsp_state* s, double* beta, double* lam_inv2, double* nu_inv, double* tau_inv2, double* xi_inv,
                  long long* sweep) {
  if (!s) return fail(HSP_EINVAL, "state is NULL");
  const int rc = sync_status(s);
  const size_t pv = (size_t)s->p * sizeof(double);
  if (beta) CK(cudaMemcpy(beta, s->beta, pv, cudaMemcpyDefault));
  if (lam_inv2) CK(cudaMemcpy(lam_inv2, s->lam_inv2, pv, cudaMemcpyDefault));
  if (nu_inv) CK(cudaMemcpy(nu_inv, s->nu_inv, pv, cudaMemcpyDefault));
  Ctl c{};
  CK(cudaMemcpy(&c, s->ctl, sizeof(Ctl), cudaMemcpyDeviceToHost));
  if (tau_inv2) CK(cudaMemcpy(tau_inv2, &c.tau_inv2, sizeof(double), cudaMemcpyDefault));
  if (xi_inv) CK(cudaMemcpy(xi_inv, &c.xi_inv, sizeof(double), cudaMemcpyDefault));
  if (sweep) *sweep = (long long)c.sweep;
  return rc;
}

int hsp_set_state(hsp_state* s, const double* beta, const double* lam_inv2, const double* nu_inv, const double* tau_inv2,
                  const double* xi_inv, long long sweep) {
  if (!s) return fail(HSP_EINVAL, "state is NULL");
  CK(cudaStreamSynchronize(s->stream));
  const size_t pv = (size_t)s->p * sizeof(double);
  if (beta) CK(cudaMemcpy(s->beta, beta, pv, cudaMemcpyDefault));
  if (lam_inv2) CK(cudaMemcpy(s->lam_inv2, lam_inv2, pv, cudaMemcpyDefault));
  if (nu_inv) CK(cudaMemcpy(s->nu_inv, nu_inv, pv, cudaMemcpyDefault));
  char* c = reinterpret_cast<char*>(s->ctl);
  if (tau_inv2) CK(cudaMemcpy(c + offsetof(Ctl, tau_inv2), tau_inv2, sizeof(double), cudaMemcpyDefault));
  if (xi_inv) CK(cudaMemcpy(c + offsetof(Ctl, xi_inv), xi_inv, sizeof(double), cudaMemcpyDefault));
  if (sweep >= 0) {
    const unsigned long long k = (unsigned long long)sweep;
    CK(cudaMemcpy(c + offsetof(Ctl, sweep), &k, sizeof(k), cudaMemcpyHostToDevice));
    s->host_sweep = sweep;
  }
  const int zero = 0;
  CK(cudaMemcpy(c + offsetof(Ctl, status), &zero, sizeof(int), cudaMemcpyHostToDevice));
  return HSP_OK;
}

int hsp_get_xtz(const hsp_state* s, double* g) {
  if (!s || !g) return fail(HSP_EINVAL, "NULL argument");
  CK(cudaStreamSynchronize(s->stream));
  CK(cudaMemcpy(g, s->g, (size_t)s->p * sizeof(double), cudaMemcpyDefault));
  return HSP_OK;
}
int hsp_get_gram(const hsp_state* s, double* G) {
  if (!s || !G) return fail(HSP_EINVAL, "NULL argument");
  CK(cudaStreamSynchronize(s->stream));
  CK(cudaMemcpy(G, s->G, (size_t)s->p * s->p * sizeof(double), cudaMemcpyDefault));
  return HSP_OK;
}
int hsp_get_chol(const hsp_state* s, double* L) {
  if (!s || !L) return fail(HSP_EINVAL, "NULL argument");
  CK(cudaStreamSynchronize(s->stream));
  const size_t rb = (size_t)s->p * sizeof(double);
  CK(cudaMemcpy2D(L, rb, s->L, (size_t)chol_ld(s->p) * sizeof(double), rb, (size_t)s->p, cudaMemcpyDefault));
  return HSP_OK;
}

int hsp_get_fused_pass_ms(hsp_state* s, double* ms, long long* launches) {
  if (!s) return fail(HSP_EINVAL, "state is NULL");
  CK(cudaStreamSynchronize(s->stream));
  const int rc = drain_fused_events(s);
  if (rc != HSP_OK) return rc;
  if (ms) *ms = s->fused_n ? s->fused_ms_sum / (double)s->fused_n : 0.0;
  if (launches) *launches = s->fused_n;
  s->fused_ms_sum = 0.0; s->fused_n = 0;
  return HSP_OK;
}

int hsp_get_plan(const hsp_state* s, int* fused_ctas, int* chol_ctas, int* overlap, double* chol_est_us) {
  if (!s) return fail(HSP_EINVAL, "state is NULL");
  if (fused_ctas) *fused_ctas = s->plan.grid;
  if (chol_ctas) *chol_ctas = s->chol.K;
  if (overlap) *overlap = s->chol.overlap ? 1 : 0;
  if (chol_est_us) *chol_est_us = s->chol.est_us;
  return HSP_OK;
}
long long hsp_get_launch_count(const hsp_state* s) { return s ? s->launches : 0; }
const char* hsp_fused_variant(const hsp_state* s) {
  return !s ? "generic" : s->plan.variant == 1 ? "tma" : s->plan.variant == 2 ? "tma-narrow" : "generic";
}

long long hsp_dbg_chol_trace(const hsp_state* s, long long* rows, long long capacity) {
  if (!s) return fail(HSP_EINVAL, "state is NULL");
  const CholPlan& pl = s->chol;
  const long long n = (long long)pl.h_tasks.size();
  if (!rows) return n;
  if (capacity < n) return fail(HSP_EINVAL, "capacity is smaller than the number of tasks");
  CK(cudaStreamSynchronize(s->stream));
  std::vector<unsigned long long> tr((size_t)n * 4, 0ull);
  if (pl.d_trace) CK(cudaMemcpy(tr.data(), pl.d_trace, tr.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost));
  std::vector<int> cta_of((size_t)n, 0);
  for (long long q = 0; q < n; ++q) {
    const CholTask& t = pl.h_tasks[(size_t)q];
    long long* r = rows + 12 * q;
    r[0] = t.type; r[1] = t.i; r[2] = t.j; r[3] = t.kbeg; r[4] = t.kend; r[5] = t.slot_in; r[6] = t.slot_out;
    r[7] = (long long)tr[4 * q + 3]; r[8] = (long long)tr[4 * q]; r[9] = (long long)tr[4 * q + 1]; r[10] = (long long)tr[4 * q + 2];
    r[11] = 0;
    if (t.type >= 2) {   // chain tasks run on CTA 0; the device keeps their end time in the last trace word
      r[7] = 0; r[10] = (long long)tr[4 * q + 3];
      if (t.type == 2) r[11] = (long long)tr[4 * q + 2];   // POTRF: r[9] = end of the tile factorisation, r[11] = end of the inverse
    }
  }
  return n;
}

long long hsp_dbg_chol_schedule(int nt, int sb, int K, int* rows, long long capacity, double* makespan_us) {
  if (nt < 1 || sb < 1 || K < 1 || (long long)K > (long long)nt * nt) return fail(HSP_EINVAL, "hsp_dbg_chol_schedule: need nt, sb >= 1 and 1 <= K <= nt^2");
  const CholSchedule sc = chol_build_schedule(nt, sb > nt ? nt : sb, K);
  const long long n = (long long)sc.tasks.size();
  if (makespan_us) *makespan_us = sc.makespan_us;
  if (!rows) return n;
  if (capacity < n) return fail(HSP_EINVAL, "capacity is smaller than the number of tasks");
  for (int k = 0; k < sc.K; ++k)
    for (int q = sc.list_off[k]; q < sc.list_off[k + 1]; ++q) {
      const CholTask& t = sc.tasks[(size_t)q];
      int* r = rows + 8 * (size_t)q;
      r[0] = k; r[1] = t.type; r[2] = t.i; r[3] = t.j; r[4] = t.kbeg; r[5] = t.kend; r[6] = t.slot_in; r[7] = t.slot_out;
    }
  return n;
}

// ---- device unit-test hooks ----------------------------------------------------------------------
__global__ void dbg_philox_kernel(const unsigned* ctr, const unsigned* key, unsigned* out, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  U4 c{ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3]};
  const U4 r = philox4x32_10(c, key[2 * i], key[2 * i + 1]);
  out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
}
__global__ void dbg_uniform_kernel(unsigned long long seed, const unsigned long long* idx, unsigned sweep, unsigned tag,
                                   double* ua, double* ub, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const U4 r = variate_bits(seed, idx[i], sweep, tag);
  if (ua) ua[i] = bits_to_unit(r.x, r.y);
  if (ub) ub[i] = bits_to_unit(r.z, r.w);
}
__global__ void dbg_tnpos_kernel(const double* m, const double* u, double* w, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const bool ok = i < n;
  const double r = tnpos(ok ? m[i] : 0.0, ok ? u[i] : 0.5);   // all lanes call: the tail vote is warp-wide
  if (ok) w[i] = r;
}
__global__ void dbg_norm_inv_kernel(const double* u, double* x, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) x[i] = norm_inv(u[i]);
}
__global__ void dbg_cheng_kernel(double alpha, unsigned long long seed, unsigned sweep0, double* x, long long n) {
  const long long w = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (w >= n) return;   // warp-uniform
  const double r = cheng_gamma_warp(alpha, seed, sweep0 + (unsigned)w);
  if ((threadIdx.x & 31) == 0) x[w] = r;
}

int hsp_dbg_philox(const unsigned* ctr, const unsigned* key, unsigned* out, long long n, void* stream) {
  if (n <= 0) return HSP_OK;
  dbg_philox_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(ctr, key, out, n);
  CK(cudaGetLastError());
  return HSP_OK;
}
int hsp_dbg_uniform(unsigned long long seed, const unsigned long long* idx, unsigned sweep, unsigned tag, double* ua,
                    double* ub, long long n, void* stream) {
  if (n <= 0) return HSP_OK;
  dbg_uniform_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(seed, idx, sweep, tag, ua, ub, n);
  CK(cudaGetLastError());
  return HSP_OK;
}
int hsp_dbg_tnpos(const double* m, const double* u, double* w, long long n, void* stream) {
  if (n <= 0) return HSP_OK;
  dbg_tnpos_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(m, u, w, n);
  CK(cudaGetLastError());
  return HSP_OK;
}
int hsp_dbg_norm_inv(const double* u, double* x, long long n, void* stream) {
  if (n <= 0) return HSP_OK;
  dbg_norm_inv_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(u, x, n);
  CK(cudaGetLastError());
  return HSP_OK;
}
int hsp_dbg_cheng(double alpha, unsigned long long seed, unsigned sweep0, double* x, long long n, void* stream) {
  if (n <= 0) return HSP_OK;
  dbg_cheng_kernel<<<(unsigned)((n * 32 + 255) / 256), 256, 0, (cudaStream_t)stream>>>(alpha, seed, sweep0, x, n);
  CK(cudaGetLastError());
  return HSP_OK;
}

}  // extern "C"

// hsp_internal.h -- host-side declarations shared by the translation units of libhsp.so.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <vector>

namespace hsp {

// Device-resident control block: everything a captured CUDA graph must read at replay time.
struct Ctl {
  unsigned long long sweep;      // number of completed sweeps k
  unsigned long long hist_base;  // sweep count when the current hsp_sweep call started
  double tau_inv2;               // tau^-2
  double xi_inv;                 // xi^-1
  int status;                    // 0, or HSP_ENOTPD / HSP_ENUMERIC (first error wins)
  int done;                      // CTAs of beta_gemv2_kernel that have finished (the last one advances `sweep`)
  double* h_beta;                // device history of the current hsp_sweep call (may be null)
  double* h_lambda;
  double* h_tau;
};

enum { kF32 = 0, kF64 = 1 };

// Plan-time options (hsp_set_option, include/hsp.h): -1 = automatic.  A chain copies the process defaults at create.
struct Options {
  int fused_eta = -1;      // eta-phase arithmetic for fp32 X: 0 exact fp64, 2 fp32 chains (default)
  int fused_grid = -1;     // CTAs of the fused pass
  int fused_stages = -1;   // ring depth S
  int fused_lag = -1;      // tiles between the eta phase and the x*z phase, D
  int fused_w = -1;        // compute threads across a row (256 / 512) for rows of 257..512 16-byte vectors
  int narrow_rt = -1;      // rows per tile of the narrow kernel
  int fused_variant = -1;  // 0 forces the generic kernel, 1 allows the TMA kernel below 128 vectors per row
  int fused_narrow = -1;   // 0 disables the narrow kernel
  int chol_ctas = -1;      // CTAs (SMs) of the Cholesky branch
  int chol_sb = -1;        // tiles per inverse super-block
  int chol_trace = -1;     // 1: per-task device timestamps (hsp_dbg_chol_trace)
  int gram_tc = -1;        // 0 / 1 forces the exact / tensor-core Gram
  int no_pdl = -1;         // 1: launch the tail kernels without programmatic dependent launch
};
inline int opt_or(int v, int dflt) { return v >= 0 ? v : dflt; }

struct FusedPlan {
  int variant;        // 0 = generic, 1 = tma (wide rows), 2 = tma-narrow (chunks = U bytes per load of the row dot product, width = skew shift)
  int grid, block;
  size_t smem;
  int rows_per_tile;  // R
  int stages;         // S
  int lag;            // D
  int chunks;         // C: 16-byte column chunks per compute thread
  int width;          // W: compute threads across one row (256 or 512)
  int groups;         // G: row groups of compute warps (partial rows = grid * G)
  int eta_mode;       // EM: arithmetic of the eta phase for fp32 X (fused_pass.cu)
  long long n_tiles;
  long long row_offset;   // global index of local row 0 (row-sharded chains: the Philox counter of z_i is the GLOBAL row)
};

// ---- fused pass (a1-a3) and reduce (b): fused_pass.cu
FusedPlan fused_plan(int dtype, long long N, int p, int num_sms, const void* X, const Options& opt);   // num_sms: CTAs the pass may use
cudaError_t fused_pass_launch(const FusedPlan& plan, const void* X, int dtype, const unsigned char* y, long long N,
                              int p, unsigned long long seed, const double* beta, const Ctl* ctl, double* partial,
                              double* z_out, cudaStream_t st);
cudaError_t reduce_partials_launch(const double* partial, int n_part, int p, double* g, cudaStream_t st);

// ---- the paper's own decomposition of a1-a3 (two products + rejection sampler), for the A/B: paper_design.cu
int paper_design_ctas(long long N, int num_sms);
cudaError_t paper_design_launch(const void* X, int dtype, const unsigned char* y, long long N, int p, unsigned long long seed,
                                const double* beta, const Ctl* ctl, double* mu, double* z, double* partial, int n_part,
                                int num_sms, cudaStream_t st);

// ---- Gram (c0): gram.cu
struct GramPlan { int slots, chunks, slots_per_chunk; long long rows_per_slot; bool tensor_core; };
GramPlan gram_plan(long long N, int p, int dtype, int num_sms, bool tensor_core);
// fp32 X on the tcgen05 tensor cores (split-bf16, fp64 flush): gram_tc.cu
cudaError_t gram_tc_chunk_launch(const GramPlan& g, int chunk, const float* X, long long N, int p, double* scratch, cudaStream_t st);
cudaError_t gram_chunk_launch(const GramPlan& g, int chunk, const void* X, int dtype, long long N, int p, double* scratch,
                              cudaStream_t st);
cudaError_t gram_finish_launch(const GramPlan& g, int p, const double* scratch, double* G, cudaStream_t st);

// ---- Q build (c), Cholesky + inverse factor (d1), beta draw (d2): cholesky.cu, chol_schedule.cu
// One tile task of the Cholesky task graph (64x64 tiles).  type 0: tile L(i,j), i >= j; type 1: inverse tile
// W(j,i), i < j.  The task accumulates k in [kbeg, kend); slot_in >= 0: start from the partial accumulator in
// that workspace slot (else from the Q tile / zero); slot_out >= 0: store the partial accumulator there
// instead of finalising the tile.  Types 2, 3, 4: the chain tasks POTRF(j), TRSM(j) -> L(j+1,j), SYRK(j) -> A(j+1,j+1) of
// the dedicated chain CTA (first list, schedules with K >= 2).
struct CholTask { int type, i, j, kbeg, kend, slot_in, slot_out, pad; };
struct CholSchedule {
  int K = 0, n_slots = 0;
  double makespan_us = 0.0;          // cost-model estimate
  std::vector<CholTask> tasks;       // concatenated per-CTA lists
  std::vector<int> list_off;         // K + 1 offsets into tasks
};
CholSchedule chol_build_schedule(int nt, int sb_tiles, int K);

struct CholPlan {
  int p = 0, nt = 0, P = 0, K = 0, n_slots = 0, n_tasks = 0;
  int sb = 0;                        // tiles per inverse super-block (sb == nt: the whole inverse factor is built)
  bool overlap = false;              // the branch is expected to hide behind the fused pass on K SMs of its own
  double est_us = 0.0;
  CholTask* d_tasks = nullptr;
  int* d_list_off = nullptr;
  int* d_flags = nullptr;            // [nt*nt] L tiles, [nt*nt] inverse tiles, [n_slots] partials
  size_t n_flags = 0;
  double* d_ws = nullptr;            // n_slots x 4096 doubles
  unsigned long long* d_trace = nullptr;   // option chol_trace = 1: four words per task: start, end of the k-loop, end (ns), CTA (chain tasks: see hsp.h)
  std::vector<CholTask> h_tasks;     // host copy of the schedule (for hsp_dbg_chol_trace)
};
int chol_tiles(int p);                 // nt = ceil(p / 64)
int chol_ld(int p);                    // P = 64 nt: leading dimension of L, W, Wt (padded with the identity)
cudaError_t chol_plan_create(CholPlan* plan, int p, int num_sms, double fused_ms_estimate, const Options& opt);
void chol_plan_destroy(CholPlan* plan);
cudaError_t cholesky_launch(const CholPlan& plan, const double* G, const double* lam_inv2, Ctl* ctl, double* L, double* W,
                            double* Wt, double* Lt, cudaStream_t st, long long* launches);
cudaError_t beta_solve_launch(const double* W, const double* Wt, const double* g, double* tv, double* beta, int p,
                              unsigned long long seed, Ctl* ctl, cudaStream_t st, long long* launches, bool pdl);
// block substitution with a block-diagonal inverse (sb < nt); rv: scratch of P doubles
cudaError_t beta_block_solve_launch(const double* L, const double* Lt, const double* W, const double* Wt, const double* g,
                                    double* tv, double* rv, double* beta, int p, int sb, unsigned long long seed, Ctl* ctl,
                                    cudaStream_t st, long long* launches, bool pdl);
cudaError_t beta_keep_launch(const double* beta, int p, Ctl* ctl, cudaStream_t st);

// ---- scale conditionals (e1, e2, e3) and draw output (g): scales.cu
cudaError_t scales_launch(const double* beta, double* lam_inv2, double* nu_inv, Ctl* ctl, int p, unsigned long long seed,
                          int freeze_scales, cudaStream_t st);
cudaError_t set_history_launch(Ctl* ctl, unsigned long long hist_base, double* hb, double* hl, double* ht, cudaStream_t st);
cudaError_t validate_y_launch(const unsigned char* y, long long N, int* bad, cudaStream_t st);
cudaError_t side_launch(const unsigned char* y, long long N, signed char* side, cudaStream_t st);

}  // namespace hsp

// Internal declarations shared by the translation units of libspd_b200.so.
// Nothing here is part of the public C ABI (include/spd.h).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/spd.h"

namespace spd {

// Dyadic-tree geometry: a block of T threads owns "rows" of 4*T consecutive
// samples, R rows per streaming step ("chunk"); T and R are chosen in spd_tree.cu.
constexpr int kTreeMaxLevels = 16;  // widths 1 .. 32768
constexpr int kStages = 3;          // bulk-copy ring depth

struct TreeConfig {
    int K = 0;            // number of widths: 2^0 .. 2^(K-1)
    int kind = 0;         // 0: block per stream (spd_tree.cu), 1: warp per stream (spd_tree_ws.cuh)
    bool ig = false;      // warp per stream: the IGRID depth-1 width set (2^k and 3 * 2^m) over the K levels
    int T = 0;            // threads per block
    int chunk = 0;        // 4 * T * R samples
    int act_block = 0;    // samples per activity-map byte (0: = chunk)
    int warm_chunks = 0;  // look-ahead chunks an interior segment replays
    int segs_per_row = 1;
    int seg_chunks = 0;   // chunks per segment
    int chunks_per_row = 0;
    int blocks_per_sm = 0;
    size_t smem_bytes = 0;
};

// Alg. 1's own widths on Alg. 1's own grids (spd_boxdit.cu); B = 0: not such a plan.
struct BoxditConfig {
    int B = 0;             // L_max per iteration (4, 8, 16 or 32; D = 2)
    int levels = 0;        // iterations
    int last_count = 0;    // widths of the last iteration (max_width may cut it)
    int chunks_per_row = 0, segs_per_row = 1, seg_chunks = 0, warm_chunks = 0;
    int smem_bytes = 0;
};

// Per-width boxcar separation (spd_plan_create_grid): consecutive widths of equal separation.
constexpr int kGridGroupsMax = 32;
struct GridGroups {
    int n;
    int shift[kGridGroupsMax];  // log2 of the group's separation
    int kb[kGridGroupsMax];     // first width of the group
    int ke[kGridGroupsMax];     // one past its last width
};

struct HostStaging {
    bool ready = false;
    int64_t rows_per_block = 0;
    cudaStream_t stream[2] = {nullptr, nullptr};
    float* d_plane[2] = {nullptr, nullptr};
    float* d_snr[2] = {nullptr, nullptr};
    void* d_width[2] = {nullptr, nullptr};
    float* d_mean = nullptr;
    float* d_sigma = nullptr;
    // spd_run_host_candidates
    uint8_t* d_act[2] = {nullptr, nullptr};  // activity map of one row block
    float* d_snr_full = nullptr;             // whole-plane Y for the 2-D peak stage (allocated on first use)
    spd_candidate* d_list = nullptr;         // 1-D candidates of all blocks
    spd_candidate* d_list2 = nullptr;        // after the 2-D stage
    int64_t list_cap = 0, list2_cap = 0;
    int64_t* d_counts = nullptr;             // [0] 1-D count, [1] 2-D count
    int64_t* h_counts = nullptr;             // pinned copy
};

}  // namespace spd

struct spd_plan {
    int64_t n_dm = 0, n_t = 0;
    std::vector<int32_t> widths;
    int32_t max_width = 0;
    int32_t path = 0;
    uint32_t flags = 0;      // SPD_FLAG_* of spd_plan_create_ex
    int width_bytes = 4;     // out_width element size: 4, or 1 (SPD_FLAG_WIDTH_U8)
    int segs_option = 0;     // SPD_OPT_SEGMENTS_PER_ROW (0 = automatic)
    int64_t host_rows_option = 0;  // SPD_OPT_HOST_ROWS_PER_BLOCK (0 = automatic)
    int device = 0;
    int sm_count = 0;
    // dyadic tree
    spd::TreeConfig tree;
    spd::BoxditConfig boxdit;
    // generic path
    int32_t* d_widths = nullptr;   // [n_widths]
    float* d_wscale = nullptr;     // [n_widths] 1/sqrt(L)
    double* d_prefix = nullptr;    // [n_dm][n_t + 1] running sums of (x - mu)
    double* d_blocksum = nullptr;  // [n_dm][blocks_per_row]
    int64_t generic_blocks_per_row = 0;
    std::vector<int32_t> separations;  // empty, or one power of two per width (grid plans)
    spd::GridGroups grid = {};
    int generic_tile = 0;  // > 0: tile kernel (time samples per block); 0: workspace kernels
    int generic_span = 0;  // tile + look-ahead, multiple of 64
    size_t generic_smem = 0;
    int64_t generic_tiles_per_row = 0;
    int64_t workspace_bytes = 0;
    // spd_row_stats
    void* d_stats = nullptr;  // [n_dm][stats_parts] partial moments
    int32_t* d_stats_state = nullptr;  // [n_dm][2]: converged flag, rejection passes done
    int stats_parts = 0;
    int64_t stats_part = 0;   // samples per part
    // spd_width_sigma
    void* d_wsig_partial = nullptr;  // [n_dm][parts][14] level sums
    void* d_wsig_totals = nullptr;   // [n_dm][super-blocks] totals of 8192 samples
    void* d_wsig_widths = nullptr;   // [n_widths] the plan's widths
    int wsig_parts = 0, wsig_sb_per_part = 0, wsig_sb_per_row = 0, wsig_levels = 0;
    // spd_run_host
    spd::HostStaging host;
};

namespace spd {

void set_error(const char* fmt, ...);
int cuda_fail(cudaError_t e, const char* what);

// spd_tree.cu
bool tree_applicable(const std::vector<int32_t>& widths, int64_t n_t);
int tree_configure(spd_plan* plan);
int tree_configure_segments(spd_plan* plan);
// activity: nullptr, or [n_dm][chunks_per_row] bytes (cleared here, set by the kernel for
// every chunk whose best SNR reaches `threshold`).
// sigma_w: nullptr (eq. 5), or [n_dm][K] measured standard deviations per width (then sigma is not read)
int tree_run(const spd_plan* plan, int64_t n_dm, const float* plane, const float* mean,
             const float* sigma, float* out_snr, void* out_width, float threshold,
             uint8_t* activity, cudaStream_t stream, const float* sigma_w = nullptr);

// spd_tree_ws.cu: the dyadic tree with one warp per stream (tensor-memory delay lines)
bool ws_applicable(int K, uint32_t flags);
int ws_configure(spd_plan* plan);
int ws_grid_blocks(const spd_plan* plan);
int ws_piece_chunks(const spd_plan* plan);
// sigma_w: nullptr (eq. 5), or [n_dm][K] measured standard deviations per width (then sigma is not read)
int ws_run(const spd_plan* plan, int64_t n_dm, const float* plane, const float* mean, const float* sigma,
           float* out_snr, void* out_width, float threshold, uint8_t* activity, cudaStream_t stream,
           const float* sigma_w = nullptr);

// spd_tree_ws_ig.cu: the warp-per-stream kernel for widths 2^k and 3 * 2^m (IGRID depth 1); plan->tree.K, .ig set
int ws_ig_configure(spd_plan* plan);
int ws_ig_run(const spd_plan* plan, int64_t n_dm, const float* plane, const float* mean, const float* sigma,
              float* out_snr, void* out_width, float threshold, uint8_t* activity, cudaStream_t stream,
              const float* sigma_w);

// spd_tree_ig.cu: widths 2^k and 3 * 2^m (IGRID depth 1)
int ig_applicable(const std::vector<int32_t>& widths, int64_t n_t);  // K (pow-2 levels) or 0
int ig_configure(spd_plan* plan);
int ig_run(const spd_plan* plan, int64_t n_dm, const float* plane, const float* mean,
           const float* sigma, float* out_snr, int32_t* out_width, float threshold,
           uint8_t* activity, cudaStream_t stream, const float* sigma_w = nullptr);

inline bool is_tree_path(const spd_plan* plan) {
    return plan->path == SPD_PATH_DYADIC_TREE || plan->path == SPD_PATH_IGRID_TREE;
}
// A streaming-tree kernel runs this plan (fused threshold test, activity map per tree.act_block / chunk):
// the tree paths, and a grid plan over widths 2^k (warp-per-stream kernel with per-level grids).
inline bool runs_tree_kernel(const spd_plan* plan) {
    return is_tree_path(plan) || (plan->path == SPD_PATH_GRID && plan->tree.kind == 1);
}

// spd_generic.cu
int generic_configure(spd_plan* plan);
void generic_release(spd_plan* plan);
// output separated by iteration (grid plans): planes of the groups of equal separation, concatenated
int64_t grid_iter_points(const spd_plan* plan, int g);
int generic_run_iterations(const spd_plan* plan, const float* plane, const float* mean, const float* sigma,
                           float* out_snr, int32_t* out_width, cudaStream_t stream);
// sigma_w: nullptr (eq. 5: sqrt(L) sigma[d]) or [n_dm][n_widths] measured standard deviations
// (tile kernels only); then `sigma` is not read.
int generic_run(const spd_plan* plan, int64_t n_dm, const float* plane, const float* mean,
                const float* sigma, float* out_snr, int32_t* out_width, cudaStream_t stream,
                const float* sigma_w = nullptr);

// spd_dense.cu: any width set with max_width <= 64 (running sums in registers)
bool dense_applicable(const spd_plan* plan);
int dense_blocks(const spd_plan* plan);
int dense_run(const spd_plan* plan, int64_t n_dm, const float* plane, const float* mean, const float* sigma,
              float* out_snr, int32_t* out_width, cudaStream_t stream, const float* sigma_w);

// spd_boxdit.cu: the BoxDIT algorithm (widths of eq. 14 on their own grids) as one streaming kernel
bool boxdit_configure(spd_plan* plan);
int boxdit_run_iterations(const spd_plan* plan, const float* plane, const float* mean, const float* sigma,
                          float* it_snr, int32_t* it_width, cudaStream_t stream);
// activity: nullptr, or [n_dm][ceil(n_t / 4096)] bytes, cleared here and set for every 4096-sample chunk with a key
// that reaches `threshold` (row a8's threshold test fused, as the tree kernels do)
int boxdit_run(const spd_plan* plan, int64_t n_dm, const float* plane, const float* mean, const float* sigma,
               float* out_snr, int32_t* out_width, cudaStream_t stream, const float* sigma_w, float threshold = 0.f,
               uint8_t* activity = nullptr);

// spd_stats.cu
int stats_configure(spd_plan* plan);
void stats_release(spd_plan* plan);
// rel_tol < 0: exactly n_iter rejection passes; else stop a row once a pass changes neither estimate by
// more than rel_tol * sigma (device-side test); n_passes: nullptr or [n_dm] rejection passes done.
int stats_run(const spd_plan* plan, const float* plane, float clip, int n_iter, float rel_tol, float* mean,
              float* sigma, int32_t* n_passes, cudaStream_t stream);

// spd_width_sigma.cu: standard deviation per width from power-of-two decimations
int wsig_configure(spd_plan* plan);
void wsig_release(spd_plan* plan);
int wsig_run(const spd_plan* plan, const float* plane, const float* mean, float* sigma_w, cudaStream_t stream);

// spd_candidates.cu
// activity: nullptr (visit every sample) or the map written by spd_run_flagged, one byte
// per `act_block` samples of each row (`act_per_row` bytes per row).
// The planes hold n_rows rows whose first is DM trial dm_offset (candidates carry dm_offset + row);
// clear: zero *n_found first (false: append to a list other launches are filling too).
int candidates_run(const spd_plan* plan, int64_t n_rows, int64_t dm_offset, const float* out_snr,
                   const void* out_width, const uint8_t* activity, float threshold, spd_candidate* list,
                   int64_t capacity, int64_t* n_found, bool clear, cudaStream_t stream);
// 2-D peak stage over a candidate list (reading A18); out_snr is the whole plane.
int cluster_run(const spd_plan* plan, const float* out_snr, const spd_candidate* list_in, const int64_t* n_in,
                int64_t capacity_in, int dm_radius, spd_candidate* list_out, int64_t capacity_out, int64_t* n_out,
                cudaStream_t stream);

// Activity-map geometry of a plan (both paths): samples per byte and bytes per row.
int64_t activity_block(const spd_plan* plan);
int64_t activity_per_row(const spd_plan* plan);

}  // namespace spd

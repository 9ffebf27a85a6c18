// Host entry points of the warp-per-stream tree kernel (spd_tree_ws.cuh) for widths {1, 2, ..., 2^(K-1)},
// 9 <= K <= 14; the IGRID depth-1 family is instantiated in spd_tree_ws_ig.cu.
#include "spd_tree_ws.cuh"

namespace spd {

// Warp-stream kernel for this plan?  Yes for kWsMinK <= K <= kWsMaxK unless the plan was created with
// SPD_FLAG_BLOCK_TREE (A/B runs against the block-per-stream kernels of spd_tree.cu / spd_tree_ig.cu).
bool ws_applicable(int K, uint32_t flags) {
    return K >= kWsMinK && K <= kWsMaxK && !(flags & SPD_FLAG_BLOCK_TREE);
}

int ws_configure(spd_plan* plan) { return plan->tree.ig ? ws_ig_configure(plan) : ws_configure_t<false>(plan); }

int ws_piece_chunks(const spd_plan* plan) {
    int pc = 0;
    int64_t np = 0;
    ws_pieces(plan, plan->n_dm, &pc, &np);
    return pc;
}

int ws_grid_blocks(const spd_plan* plan) {
    int pc = 0;
    int64_t np = 0;
    ws_pieces(plan, plan->n_dm, &pc, &np);
    return static_cast<int>(std::max<int64_t>(1, std::min<int64_t>(plan->sm_count, (np + kWsWarps - 1) / kWsWarps)));
}

int ws_run(const spd_plan* plan, int64_t n_dm, const float* plane, const float* mean, const float* sigma,
           float* out_snr, void* out_width, float threshold, uint8_t* activity, cudaStream_t stream,
           const float* sigma_w) {
    if (plan->tree.ig)
        return ws_ig_run(plan, n_dm, plane, mean, sigma, out_snr, out_width, threshold, activity, stream, sigma_w);
    return ws_run_t<false>(plan, n_dm, plane, mean, sigma, out_snr, out_width, threshold, activity, stream, sigma_w);
}

}  // namespace spd

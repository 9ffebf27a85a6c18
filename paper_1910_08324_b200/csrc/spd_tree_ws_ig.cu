// The warp-per-stream tree kernel (spd_tree_ws.cuh) instantiated for the IGRID depth-1 width set: widths 2^k
// and 3 * 2^m up to 2^(K-1), 9 <= K <= 14 (eq. 18 / Table 1).  Its own translation unit so
// that the two families compile in parallel.
#include "spd_tree_ws.cuh"

namespace spd {

int ws_ig_configure(spd_plan* plan) { return ws_configure_t<true>(plan); }

int ws_ig_run(const spd_plan* plan, int64_t n_dm, const float* plane, const float* mean, const float* sigma,
              float* out_snr, void* out_width, float threshold, uint8_t* activity, cudaStream_t stream,
              const float* sigma_w) {
    return ws_run_t<true>(plan, n_dm, plane, mean, sigma, out_snr, out_width, threshold, activity, stream, sigma_w);
}

}  // namespace spd

// C ABI of libspd_b200.so (include/spd.h): plans, width-set generators, dispatch,
// the host-buffer entry point and error reporting.  All compute is in the kernels of
// spd_tree.cu / spd_generic.cu / spd_candidates.cu; there is no CPU fallback.
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <new>

#include "spd_internal.h"

namespace spd {

static thread_local char g_error[512] = "";

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_error, sizeof(g_error), fmt, ap);
    va_end(ap);
}

int cuda_fail(cudaError_t e, const char* what) {
    set_error("CUDA error while %s: %s (%s)", what, cudaGetErrorName(e), cudaGetErrorString(e));
    cudaGetLastError();  // clear the sticky-free error state
    return SPD_ERR_CUDA;
}

namespace {

// ---- width sets ------------------------------------------------------------------------
// ALL: PAPER.md:193.  POW2: PAPER.md:311.  BOXDIT: eq. (14), D = 2 - iteration i
// covers (2^i - 1) L_max + 2^i m, m = 1..L_max (example L_max = 4: 1,2,3,4 then 6,8,10,12,
// PAPER.md:201).  IGRID: eq. (18) / Table 1, PAPER.md:364-387 - octave 2^i contributes
// 2^i + j 2^(i-depth), j = 0 .. 2^depth - 1 (16 -> 16,24 | 16,20,24,28 | 16,18,..,30).
int generate_widths(int32_t kind, int32_t param, int32_t max_width, std::vector<int32_t>& w) {
    w.clear();
    if (max_width < 1) {
        set_error("max_width must be >= 1 (got %d)", max_width);
        return SPD_ERR_INVALID_ARG;
    }
    switch (kind) {
        case SPD_WIDTHS_ALL:
            for (int64_t L = 1; L <= max_width; ++L) w.push_back(static_cast<int32_t>(L));
            break;
        case SPD_WIDTHS_POW2:
            for (int64_t L = 1; L <= max_width; L *= 2) w.push_back(static_cast<int32_t>(L));
            break;
        case SPD_WIDTHS_BOXDIT: {
            if (param < 1) {
                set_error("BOXDIT needs param = L_max >= 1 (got %d)", param);
                return SPD_ERR_INVALID_ARG;
            }
            for (int i = 0; i < 31; ++i) {
                const int64_t step = int64_t(1) << i;
                const int64_t base = (step - 1) * param;
                if (base >= max_width) break;
                for (int64_t m = 1; m <= param; ++m) {
                    const int64_t L = base + step * m;
                    if (L > max_width) break;
                    w.push_back(static_cast<int32_t>(L));
                }
            }
            break;
        }
        case SPD_WIDTHS_IGRID: {
            if (param < 0 || param > 16) {
                set_error("IGRID needs 0 <= param = depth <= 16 (got %d)", param);
                return SPD_ERR_INVALID_ARG;
            }
            for (int64_t oct = 1; oct <= max_width; oct *= 2) {
                const int64_t step = std::max<int64_t>(1, oct >> param);
                for (int64_t L = oct; L < 2 * oct && L <= max_width; L += step) w.push_back(static_cast<int32_t>(L));
            }
            break;
        }
        case SPD_WIDTHS_GEOMETRIC: {
            if (param <= 1000) {
                set_error("GEOMETRIC needs param = 1000 * ratio > 1000 (got %d)", param);
                return SPD_ERR_INVALID_ARG;
            }
            const double r = param / 1000.0;
            for (double x = 1.0; nearbyint(x) <= max_width; x *= r) w.push_back(static_cast<int32_t>(nearbyint(x)));
            break;
        }
        default:
            set_error("unknown width-set kind %d", kind);
            return SPD_ERR_INVALID_ARG;
    }
    std::sort(w.begin(), w.end());
    w.erase(std::unique(w.begin(), w.end()), w.end());
    return SPD_OK;
}

int check_device(int* device, int* sm_count) {
    cudaError_t e = cudaGetDevice(device);
    if (e != cudaSuccess) {
        set_error("no usable CUDA device: %s (this library has no CPU fallback)", cudaGetErrorString(e));
        cudaGetLastError();
        return SPD_ERR_UNSUPPORTED_DEVICE;
    }
    int major = 0;
    if ((e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, *device)) != cudaSuccess ||
        (e = cudaDeviceGetAttribute(sm_count, cudaDevAttrMultiProcessorCount, *device)) != cudaSuccess) {
        set_error("cannot query the CUDA device: %s", cudaGetErrorString(e));
        cudaGetLastError();
        return SPD_ERR_UNSUPPORTED_DEVICE;
    }
    if (major != 10) {
        set_error("device compute capability %d.x is not supported: this library is built for sm_100a only", major);
        return SPD_ERR_UNSUPPORTED_DEVICE;
    }
    return SPD_OK;
}

void release_host_staging(spd_plan* plan) {
    HostStaging& h = plan->host;
    for (int i = 0; i < 2; ++i) {
        cudaFree(h.d_plane[i]);
        cudaFree(h.d_snr[i]);
        cudaFree(h.d_width[i]);
        if (h.stream[i]) cudaStreamDestroy(h.stream[i]);
        h.d_plane[i] = nullptr;
        h.d_snr[i] = nullptr;
        h.d_width[i] = nullptr;
        h.stream[i] = nullptr;
    }
    for (int i = 0; i < 2; ++i) {
        cudaFree(h.d_act[i]);
        h.d_act[i] = nullptr;
    }
    cudaFree(h.d_mean);
    cudaFree(h.d_sigma);
    cudaFree(h.d_snr_full);
    cudaFree(h.d_list);
    cudaFree(h.d_list2);
    cudaFree(h.d_counts);
    if (h.h_counts) cudaFreeHost(h.h_counts);
    h.d_mean = h.d_sigma = h.d_snr_full = nullptr;
    h.d_list = h.d_list2 = nullptr;
    h.d_counts = h.h_counts = nullptr;
    h.list_cap = h.list2_cap = 0;
    h.ready = false;
}

int prepare_host_staging(spd_plan* plan) {
    HostStaging& h = plan->host;
    if (h.ready) return SPD_OK;
    // Row blocks of about 256 MiB of input: large enough to run the device near its
    // streaming rate, small enough that two of them (double buffering) cost 1.5 GiB.
    const int64_t row_bytes = plan->n_t * 4;
    h.rows_per_block = std::max<int64_t>(1, std::min<int64_t>(plan->n_dm, (int64_t(256) << 20) / row_bytes));
    if (plan->host_rows_option > 0) h.rows_per_block = std::min<int64_t>(plan->n_dm, plan->host_rows_option);
    const size_t elems = static_cast<size_t>(h.rows_per_block) * static_cast<size_t>(plan->n_t);
    cudaError_t e = cudaSuccess;
    for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
        if ((e = cudaStreamCreateWithFlags(&h.stream[i], cudaStreamNonBlocking)) != cudaSuccess) break;
        if ((e = cudaMalloc(&h.d_plane[i], elems * 4)) != cudaSuccess) break;
        if ((e = cudaMalloc(&h.d_snr[i], elems * 4)) != cudaSuccess) break;
        if ((e = cudaMalloc(&h.d_width[i], elems * plan->width_bytes)) != cudaSuccess) break;
    }
    if (e == cudaSuccess) e = cudaMalloc(&h.d_mean, sizeof(float) * plan->n_dm);
    if (e == cudaSuccess) e = cudaMalloc(&h.d_sigma, sizeof(float) * plan->n_dm);
    if (e != cudaSuccess) {
        set_error("allocating the host-run staging buffers failed: %s", cudaGetErrorString(e));
        cudaGetLastError();
        release_host_staging(plan);
        return SPD_ERR_ALLOC;
    }
    h.ready = true;
    return SPD_OK;
}

// Rows a1-a7 (+ the threshold test of a8 when activity != nullptr) over n_rows rows.
int run_rows(const spd_plan* plan, int64_t n_rows, const float* plane, const float* mean, const float* sigma,
             float* out_snr, void* out_width, float threshold, uint8_t* activity, cudaStream_t stream) {
    if (plan->path == SPD_PATH_DYADIC_TREE)
        return tree_run(plan, n_rows, plane, mean, sigma, out_snr, out_width, threshold, activity, stream);
    if (plan->path == SPD_PATH_IGRID_TREE && plan->tree.kind == 1)
        return ws_run(plan, n_rows, plane, mean, sigma, out_snr, out_width, threshold, activity, stream);
    if (plan->path == SPD_PATH_IGRID_TREE)
        return ig_run(plan, n_rows, plane, mean, sigma, out_snr, static_cast<int32_t*>(out_width), threshold, activity,
                      stream);
    if (plan->path == SPD_PATH_GRID && plan->tree.kind == 1)
        return ws_run(plan, n_rows, plane, mean, sigma, out_snr, out_width, threshold, activity, stream);
    if (plan->boxdit.B > 0 && plan->width_bytes == 4)  // the BoxDIT streaming kernel fuses the threshold test as well
        return boxdit_run(plan, n_rows, plane, mean, sigma, out_snr, static_cast<int32_t*>(out_width), stream, nullptr,
                          threshold, activity);
    if (activity) {
        // any-width-set path: no fused test, every block stays active (padding included: the
        // candidate kernel bounds the flag index itself)
        const size_t bytes = (static_cast<size_t>(n_rows) * static_cast<size_t>(activity_per_row(plan)) + 127) / 128 * 128;
        const cudaError_t e = cudaMemsetAsync(activity, 1, bytes, stream);
        if (e != cudaSuccess) return cuda_fail(e, "filling the activity map");
    }
    return generic_run(plan, n_rows, plane, mean, sigma, out_snr, static_cast<int32_t*>(out_width), stream);
}

size_t activity_bytes_rows(const spd_plan* plan, int64_t rows) {
    return (static_cast<size_t>(rows) * static_cast<size_t>(activity_per_row(plan)) + 127) / 128 * 128;
}
size_t activity_bytes(const spd_plan* plan) { return activity_bytes_rows(plan, plan->n_dm); }

bool misaligned16(const void* a, const void* b, const void* c) {
    return ((reinterpret_cast<uintptr_t>(a) | reinterpret_cast<uintptr_t>(b) | reinterpret_cast<uintptr_t>(c)) & 15u) != 0;
}

}  // namespace
}  // namespace spd

using namespace spd;

extern "C" {

int spd_version(void) { return SPD_VERSION; }

const char* spd_last_error_string(void) { return g_error; }

int spd_width_set_generate(int32_t kind, int32_t param, int32_t max_width, int32_t* out, int32_t cap,
                           int32_t* n_out) {
    if (!n_out || cap < 0 || (cap > 0 && !out)) {
        set_error("spd_width_set_generate: NULL output or negative capacity");
        return SPD_ERR_INVALID_ARG;
    }
    std::vector<int32_t> w;
    const int rc = generate_widths(kind, param, max_width, w);
    if (rc != SPD_OK) return rc;
    *n_out = static_cast<int32_t>(w.size());
    if (cap == 0 && !out) return SPD_OK;  // size query
    if (static_cast<size_t>(cap) < w.size()) {
        set_error("spd_width_set_generate: capacity %d < %zu widths", cap, w.size());
        return SPD_ERR_INVALID_ARG;
    }
    memcpy(out, w.data(), w.size() * sizeof(int32_t));
    return SPD_OK;
}

int spd_plan_create(spd_plan** out, int64_t n_dm, int64_t n_t, const int32_t* width_set, int32_t n_widths,
                    int32_t max_width) {
    return spd_plan_create_ex(out, n_dm, n_t, width_set, n_widths, max_width, 0u);
}

static int plan_create(spd_plan** out, int64_t n_dm, int64_t n_t, const int32_t* width_set,
                       const int32_t* separations, int32_t n_widths, int32_t max_width, uint32_t flags);

int spd_plan_create_ex(spd_plan** out, int64_t n_dm, int64_t n_t, const int32_t* width_set, int32_t n_widths,
                       int32_t max_width, uint32_t flags) {
    return plan_create(out, n_dm, n_t, width_set, nullptr, n_widths, max_width, flags);
}

int spd_plan_create_grid_ex(spd_plan** out, int64_t n_dm, int64_t n_t, const int32_t* width_set,
                            const int32_t* separations, int32_t n_widths, int32_t max_width, uint32_t flags) {
    if (!separations) {
        set_error("spd_plan_create_grid: separations is NULL");
        if (out) *out = nullptr;
        return SPD_ERR_INVALID_ARG;
    }
    if (flags & ~SPD_FLAG_FORCE_GENERIC) {
        set_error("spd_plan_create_grid_ex: only SPD_FLAG_FORCE_GENERIC applies to a grid plan (got 0x%x)", flags);
        if (out) *out = nullptr;
        return SPD_ERR_INVALID_ARG;
    }
    return plan_create(out, n_dm, n_t, width_set, separations, n_widths, max_width, flags);
}

int spd_plan_create_grid(spd_plan** out, int64_t n_dm, int64_t n_t, const int32_t* width_set,
                         const int32_t* separations, int32_t n_widths, int32_t max_width) {
    return spd_plan_create_grid_ex(out, n_dm, n_t, width_set, separations, n_widths, max_width, 0u);
}

int spd_separation_generate(int32_t kind, int32_t param, const int32_t* widths, int32_t n_widths, int32_t* out) {
    if (!widths || !out || n_widths < 1) {
        set_error("spd_separation_generate: NULL argument or no widths");
        return SPD_ERR_INVALID_ARG;
    }
    for (int32_t k = 0; k < n_widths; ++k) {
        const int64_t L = widths[k];
        if (L < 1) {
            set_error("spd_separation_generate: width %lld < 1", (long long)L);
            return SPD_ERR_INVALID_ARG;
        }
        int64_t oct = 1;  // largest power of two <= L
        while (oct * 2 <= L) oct *= 2;
        int64_t sep = 1;
        switch (kind) {
            case SPD_GRID_EVERY_SAMPLE:
                break;
            case SPD_GRID_DIT:  // Alg. 3: width 2^i at every 2^i-th sample
                if (oct != L) {
                    set_error("SPD_GRID_DIT needs power-of-two widths (got %lld)", (long long)L);
                    return SPD_ERR_INVALID_ARG;
                }
                sep = L;
                break;
            case SPD_GRID_BOXDIT: {  // Alg. 1 with D = 2: iteration i holds widths (2^i - 1) L_max + 2^i m (eq. 14)
                if (param < 1) {
                    set_error("SPD_GRID_BOXDIT needs param = L_max >= 1");
                    return SPD_ERR_INVALID_ARG;
                }
                int64_t base = 0, step = 1;
                while (L > base + step * param) {
                    base += step * param;
                    step *= 2;
                }
                sep = step;
                break;
            }
            case SPD_GRID_IGRID:  // P layers: L_s = 2^i / P for the widths of step 2^i
                if (param < 1 || (param & (param - 1))) {
                    set_error("SPD_GRID_IGRID needs param = number of layers, a power of two");
                    return SPD_ERR_INVALID_ARG;
                }
                sep = std::max<int64_t>(1, oct / param);
                break;
            default:
                set_error("unknown separation kind %d", kind);
                return SPD_ERR_INVALID_ARG;
        }
        out[k] = static_cast<int32_t>(sep);
    }
    return SPD_OK;
}

static int plan_create(spd_plan** out, int64_t n_dm, int64_t n_t, const int32_t* width_set,
                       const int32_t* separations, int32_t n_widths, int32_t max_width, uint32_t flags) {
    if (!out) {
        set_error("spd_plan_create: out is NULL");
        return SPD_ERR_INVALID_ARG;
    }
    *out = nullptr;
    if (n_dm < 1 || n_t < 1 || n_t > 0x7fffffffll || n_dm > 0x7fffffffll) {
        set_error("spd_plan_create: bad plane shape %lld x %lld", (long long)n_dm, (long long)n_t);
        return SPD_ERR_INVALID_ARG;
    }
    if (!width_set || n_widths < 1) {
        set_error("spd_plan_create: empty width set");
        return SPD_ERR_INVALID_ARG;
    }
    if (max_width < 1 || max_width > n_t) {
        set_error("spd_plan_create: max_width %d must be in [1, n_t = %lld]", max_width, (long long)n_t);
        return SPD_ERR_INVALID_ARG;
    }
    std::vector<int32_t> w(width_set, width_set + n_widths);
    std::vector<int32_t> seps;
    GridGroups groups = {};
    if (separations) {
        // widths strictly ascending; separations powers of two that do not decrease with the width
        // (the paper's grids: an iteration's widths share D^(i), later iterations are coarser)
        seps.assign(separations, separations + n_widths);
        for (int32_t k = 0; k < n_widths; ++k) {
            const int32_t sp = seps[k];
            if (sp < 1 || (sp & (sp - 1)) || (k > 0 && (w[k] <= w[k - 1] || sp < seps[k - 1]))) {
                set_error("spd_plan_create_grid: widths must ascend strictly, separations must be powers of two "
                          "that do not decrease (entry %d: width %d, separation %d)", k, w[k], sp);
                return SPD_ERR_INVALID_ARG;
            }
            if (k == 0 || sp != seps[k - 1]) {
                if (groups.n == kGridGroupsMax) {
                    set_error("spd_plan_create_grid: more than %d distinct separations", kGridGroupsMax);
                    return SPD_ERR_INVALID_ARG;
                }
                int sh = 0;
                while ((1 << sh) < sp) ++sh;
                groups.shift[groups.n] = sh;
                groups.kb[groups.n] = k;
                ++groups.n;
            }
            groups.ke[groups.n - 1] = k + 1;
        }
    }
    std::sort(w.begin(), w.end());
    w.erase(std::unique(w.begin(), w.end()), w.end());
    if (w.front() < 1 || w.back() > max_width) {
        set_error("spd_plan_create: widths must lie in [1, max_width = %d] (got %d .. %d)", max_width, w.front(),
                  w.back());
        return SPD_ERR_INVALID_ARG;
    }
    if (w.size() > 32768) {
        set_error("spd_plan_create: more than 32768 distinct widths");
        return SPD_ERR_INVALID_ARG;
    }
    int device = 0, sm_count = 0;
    int rc = check_device(&device, &sm_count);
    if (rc != SPD_OK) return rc;

    spd_plan* plan = new (std::nothrow) spd_plan();
    if (!plan) {
        set_error("spd_plan_create: out of host memory");
        return SPD_ERR_ALLOC;
    }
    plan->n_dm = n_dm;
    plan->n_t = n_t;
    plan->widths = w;
    plan->max_width = max_width;
    plan->device = device;
    plan->sm_count = sm_count;
    plan->separations = seps;
    plan->grid = groups;
    plan->flags = flags;
    plan->width_bytes = (flags & SPD_FLAG_WIDTH_U8) ? 1 : 4;
    if ((flags & SPD_FLAG_WIDTH_U8) &&
        (separations || (flags & SPD_FLAG_FORCE_GENERIC) || !tree_applicable(w, n_t))) {
        set_error("SPD_FLAG_WIDTH_U8 needs a width set {1, 2, 4, ..., 2^(K-1)} on the streaming tree (n_t %% 4 == 0)");
        delete plan;
        return SPD_ERR_INVALID_ARG;
    }
    int ig_levels = 0;
    if (separations) {
        plan->path = SPD_PATH_GRID;
        rc = generic_configure(plan);
        // widths {2^k} on a grid: the warp-per-stream tree kernel with the keys of a level counted only on
        // that level's grid (the any-width-set grid kernel stays configured for spd_run_sigma_w)
        int igl = 0;
        if (rc == SPD_OK && !(flags & SPD_FLAG_FORCE_GENERIC) && boxdit_configure(plan)) {
            // Alg. 1's widths on Alg. 1's grids: the BoxDIT streaming kernel (spd_boxdit.cu)
        } else if (rc == SPD_OK && !(flags & SPD_FLAG_FORCE_GENERIC) && tree_applicable(w, n_t) &&
                   ws_applicable(static_cast<int>(w.size()), 0u)) {
            plan->tree.K = static_cast<int>(w.size());
            rc = ws_configure(plan);
        } else if (rc == SPD_OK && !(flags & SPD_FLAG_FORCE_GENERIC) && (igl = ig_applicable(w, n_t)) > 0 &&
                   ws_applicable(igl, 0u)) {
            // the IGRID depth-1 widths on a grid whose octaves share a separation (the widths of
            // step 2^i on P layers): width 3 * 2^m goes with width 2^(m+1)
            bool shared = true;
            for (int m = 0; m + 2 < igl; ++m) shared = shared && seps[2 * m + 2] == seps[2 * (m + 1) - 1];
            if (shared) {
                plan->tree.K = igl;
                plan->tree.ig = true;
                rc = ws_configure(plan);
            }
        }
    } else if (!(flags & SPD_FLAG_FORCE_GENERIC) && tree_applicable(w, n_t)) {
        plan->path = SPD_PATH_DYADIC_TREE;
        rc = tree_configure(plan);
    } else if (!(flags & SPD_FLAG_FORCE_GENERIC) && (ig_levels = ig_applicable(w, n_t)) > 0) {
        plan->path = SPD_PATH_IGRID_TREE;
        plan->tree.K = ig_levels;
        if (ws_applicable(ig_levels, flags)) {
            plan->tree.ig = true;
            rc = ws_configure(plan);
        } else {
            rc = ig_configure(plan);
        }
    } else {
        plan->path = SPD_PATH_GENERIC;
        rc = generic_configure(plan);
    }
    if (rc == SPD_OK) rc = stats_configure(plan);
    if (rc == SPD_OK) rc = wsig_configure(plan);
    if (rc != SPD_OK) {
        generic_release(plan);
        stats_release(plan);
        wsig_release(plan);
        delete plan;
        return rc;
    }
    *out = plan;
    return SPD_OK;
}

void spd_plan_destroy(spd_plan* plan) {
    if (!plan) return;
    release_host_staging(plan);
    generic_release(plan);
    stats_release(plan);
    wsig_release(plan);
    delete plan;
}

void spd_destroy(spd_plan* plan) { spd_plan_destroy(plan); }

int spd_plan_set_option(spd_plan* plan, int32_t option, int64_t value) {
    if (!plan) {
        set_error("spd_plan_set_option: plan is NULL");
        return SPD_ERR_INVALID_ARG;
    }
    switch (option) {
        case SPD_OPT_SEGMENTS_PER_ROW: {
            if (plan->boxdit.B > 0 && value >= 0 && value <= 0x7fffffffll) {
                plan->segs_option = static_cast<int>(value);
                boxdit_configure(plan);
                return SPD_OK;
            }
            if (!runs_tree_kernel(plan) || value < 0 || value > 0x7fffffffll) {
                set_error("SPD_OPT_SEGMENTS_PER_ROW needs a streaming-tree plan and a value >= 0 (got %lld)",
                          static_cast<long long>(value));
                return SPD_ERR_INVALID_ARG;
            }
            const int old = plan->segs_option;
            plan->segs_option = static_cast<int>(value);
            const int rc = plan->tree.kind == 1 ? ws_configure(plan) : tree_configure_segments(plan);
            if (rc != SPD_OK) {
                plan->segs_option = old;
                if (plan->tree.kind == 1) ws_configure(plan); else tree_configure_segments(plan);
            }
            return rc;
        }
        case SPD_OPT_HOST_ROWS_PER_BLOCK:
            if (value < 0) {
                set_error("SPD_OPT_HOST_ROWS_PER_BLOCK needs a value >= 0");
                return SPD_ERR_INVALID_ARG;
            }
            plan->host_rows_option = value;
            release_host_staging(plan);
            return SPD_OK;
        default:
            set_error("spd_plan_set_option: unknown option %d", option);
            return SPD_ERR_INVALID_ARG;
    }
}

int spd_plan_get_widths(const spd_plan* plan, int32_t* out, int32_t* n) {
    if (!plan || !n) {
        set_error("spd_plan_get_widths: NULL argument");
        return SPD_ERR_INVALID_ARG;
    }
    *n = static_cast<int32_t>(plan->widths.size());
    if (out) memcpy(out, plan->widths.data(), plan->widths.size() * sizeof(int32_t));
    return SPD_OK;
}

int spd_plan_get_iterations(const spd_plan* plan, int32_t cap, int32_t* n_iter, int32_t* first_width,
                            int32_t* n_widths, int32_t* separation, int64_t* n_points) {
    if (!plan || !n_iter || cap < 0) {
        set_error("spd_plan_get_iterations: NULL argument or negative cap");
        return SPD_ERR_INVALID_ARG;
    }
    if (plan->separations.empty()) {
        set_error("spd_plan_get_iterations: the plan has no boxcar separations (create it with spd_plan_create_grid)");
        return SPD_ERR_INVALID_ARG;
    }
    *n_iter = plan->grid.n;
    for (int g = 0; g < plan->grid.n && g < cap; ++g) {
        if (first_width) first_width[g] = plan->grid.kb[g];
        if (n_widths) n_widths[g] = plan->grid.ke[g] - plan->grid.kb[g];
        if (separation) separation[g] = 1 << plan->grid.shift[g];
        if (n_points) n_points[g] = grid_iter_points(plan, g);
    }
    return SPD_OK;
}

int spd_run_iterations(const spd_plan* plan, const float* plane, const float* mean, const float* sigma,
                       float* out_snr_iter, int32_t* out_width_iter, void* cuda_stream) {
    if (!plan || !plane || !mean || !sigma || !out_snr_iter || !out_width_iter) {
        set_error("spd_run_iterations: NULL argument");
        return SPD_ERR_INVALID_ARG;
    }
    if (plan->separations.empty()) {
        set_error("spd_run_iterations: the plan has no boxcar separations (create it with spd_plan_create_grid)");
        return SPD_ERR_INVALID_ARG;
    }
    return generic_run_iterations(plan, plane, mean, sigma, out_snr_iter, out_width_iter,
                                  static_cast<cudaStream_t>(cuda_stream));
}

int spd_plan_get_info(const spd_plan* plan, spd_plan_info* info) {
    if (!plan || !info) {
        set_error("spd_plan_get_info: NULL argument");
        return SPD_ERR_INVALID_ARG;
    }
    memset(info, 0, sizeof(*info));
    info->n_dm = plan->n_dm;
    info->n_t = plan->n_t;
    info->n_widths = static_cast<int32_t>(plan->widths.size());
    info->max_width = plan->max_width;
    info->path = plan->path;
    info->width_bytes = plan->width_bytes;
    info->flags = plan->flags;
    if (runs_tree_kernel(plan)) {
        info->launches_per_run = 1;
        info->threads_per_block = plan->tree.T;
        info->blocks = plan->tree.kind == 1 ? ws_grid_blocks(plan)
                                            : static_cast<int32_t>(plan->n_dm * plan->tree.segs_per_row);
        info->chunk = plan->tree.chunk;
        info->segments_per_row = plan->tree.segs_per_row;
        info->smem_bytes = static_cast<int64_t>(plan->tree.smem_bytes);
        if (is_tree_path(plan)) info->tree_kernel = plan->tree.kind == 1 ? 2 : 1;
        if (plan->tree.kind == 1 && plan->tree.segs_per_row == 0) info->piece_chunks = ws_piece_chunks(plan);
    } else {
        if (plan->boxdit.B > 0) {
            info->launches_per_run = 1;
            info->threads_per_block = 256;
            info->blocks = static_cast<int32_t>(plan->n_dm * plan->boxdit.segs_per_row);
            info->chunk = 4096;
            info->segments_per_row = plan->boxdit.segs_per_row;
            info->smem_bytes = plan->boxdit.smem_bytes;
        } else if (plan->path == SPD_PATH_GENERIC && dense_applicable(plan)) {
            info->launches_per_run = 1;
            info->threads_per_block = 256;
            info->blocks = dense_blocks(plan);
            info->chunk = 1024;
        } else if (plan->generic_tile > 0) {
            info->launches_per_run = 1;
            info->threads_per_block = 1024;
            info->blocks = static_cast<int32_t>(plan->n_dm * plan->generic_tiles_per_row);
            info->chunk = plan->generic_tile;
            info->smem_bytes = static_cast<int64_t>(plan->generic_smem);
        } else {
            info->launches_per_run = 4;
            info->threads_per_block = 256;
            info->blocks = static_cast<int32_t>(plan->n_dm * ((plan->n_t + 255) / 256));
        }
    }
    if (plan->path == SPD_PATH_GRID && plan->tree.kind == 1) info->tree_kernel = 2;
    info->workspace_bytes = plan->workspace_bytes;
    info->activity_bytes = static_cast<int64_t>(activity_bytes(plan));
    info->activity_block = static_cast<int32_t>(activity_block(plan));
    info->activity_per_row = static_cast<int32_t>(activity_per_row(plan));
    return SPD_OK;
}

int spd_run(const spd_plan* plan, const float* plane, const float* mean, const float* sigma, float* out_snr,
            void* out_width, void* cuda_stream) {
    if (!plan || !plane || !mean || !sigma || !out_snr || !out_width) {
        set_error("spd_run: NULL argument");
        return SPD_ERR_INVALID_ARG;
    }
    if (misaligned16(plane, out_snr, out_width)) {
        set_error("spd_run: plane, out_snr and out_width must be 16-byte aligned");
        return SPD_ERR_INVALID_ARG;
    }
    return run_rows(plan, plan->n_dm, plane, mean, sigma, out_snr, out_width, 0.0f, nullptr,
                    static_cast<cudaStream_t>(cuda_stream));
}

int spd_width_sigma(const spd_plan* plan, const float* plane, const float* mean, float* sigma_w, void* cuda_stream) {
    if (!plan || !plane || !mean || !sigma_w) {
        set_error("spd_width_sigma: NULL argument");
        return SPD_ERR_INVALID_ARG;
    }
    return wsig_run(plan, plane, mean, sigma_w, static_cast<cudaStream_t>(cuda_stream));
}

int spd_run_sigma_w(const spd_plan* plan, const float* plane, const float* mean, const float* sigma_w,
                    float* out_snr, void* out_width, void* cuda_stream) {
    if (!plan || !plane || !mean || !sigma_w || !out_snr || !out_width) {
        set_error("spd_run_sigma_w: NULL argument");
        return SPD_ERR_INVALID_ARG;
    }
    if (misaligned16(plane, out_snr, out_width)) {
        set_error("spd_run_sigma_w: plane, out_snr and out_width must be 16-byte aligned");
        return SPD_ERR_INVALID_ARG;
    }
    if (plan->width_bytes != 4) {
        set_error("spd_run_sigma_w: not available for SPD_FLAG_WIDTH_U8 plans");
        return SPD_ERR_INVALID_ARG;
    }
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (plan->path == SPD_PATH_DYADIC_TREE)  // run-time scale 1 / sigma_{d, 2^k} per level
        return tree_run(plan, plan->n_dm, plane, mean, nullptr, out_snr, out_width, 0.0f, nullptr, stream, sigma_w);
    if (plan->path == SPD_PATH_IGRID_TREE && plan->tree.kind == 1)
        return ws_run(plan, plan->n_dm, plane, mean, nullptr, out_snr, out_width, 0.0f, nullptr, stream, sigma_w);
    if (plan->path == SPD_PATH_IGRID_TREE)
        return ig_run(plan, plan->n_dm, plane, mean, nullptr, out_snr, static_cast<int32_t*>(out_width), 0.0f, nullptr,
                      stream, sigma_w);
    return generic_run(plan, plan->n_dm, plane, mean, nullptr, out_snr, static_cast<int32_t*>(out_width), stream,
                       sigma_w);
}

int spd_find_candidates(const spd_plan* plan, const float* out_snr, const void* out_width, float threshold,
                        spd_candidate* list, int64_t capacity, int64_t* n_found, void* cuda_stream) {
    if (!plan || !out_snr || !out_width || !n_found || capacity < 0 || (capacity > 0 && !list)) {
        set_error("spd_find_candidates: NULL argument or negative capacity");
        return SPD_ERR_INVALID_ARG;
    }
    return candidates_run(plan, plan->n_dm, 0, out_snr, out_width, nullptr, threshold, list, capacity, n_found, true,
                          static_cast<cudaStream_t>(cuda_stream));
}

int spd_run_flagged(const spd_plan* plan, const float* plane, const float* mean, const float* sigma, float* out_snr,
                    void* out_width, float threshold, uint8_t* activity, void* cuda_stream) {
    if (!plan || !plane || !mean || !sigma || !out_snr || !out_width || !activity) {
        set_error("spd_run_flagged: NULL argument");
        return SPD_ERR_INVALID_ARG;
    }
    if (misaligned16(plane, out_snr, out_width) || misaligned16(activity, nullptr, nullptr)) {
        set_error("spd_run_flagged: plane, out_snr, out_width and activity must be 16-byte aligned");
        return SPD_ERR_INVALID_ARG;
    }
    return run_rows(plan, plan->n_dm, plane, mean, sigma, out_snr, out_width, threshold, activity,
                    static_cast<cudaStream_t>(cuda_stream));
}

int spd_find_candidates_flagged(const spd_plan* plan, const float* out_snr, const void* out_width,
                                const uint8_t* activity, float threshold, spd_candidate* list, int64_t capacity,
                                int64_t* n_found, void* cuda_stream) {
    if (!plan || !out_snr || !out_width || !activity || !n_found || capacity < 0 || (capacity > 0 && !list)) {
        set_error("spd_find_candidates_flagged: NULL argument or negative capacity");
        return SPD_ERR_INVALID_ARG;
    }
    if (misaligned16(out_snr, activity, nullptr)) {
        set_error("spd_find_candidates_flagged: out_snr and activity must be 16-byte aligned");
        return SPD_ERR_INVALID_ARG;
    }
    return candidates_run(plan, plan->n_dm, 0, out_snr, out_width, activity, threshold, list, capacity, n_found, true,
                          static_cast<cudaStream_t>(cuda_stream));
}

int spd_row_stats(const spd_plan* plan, const float* plane, float clip_sigma, int32_t n_reject_passes, float* mean,
                  float* sigma, void* cuda_stream) {
    if (!plan || !plane || !mean || !sigma) {
        set_error("spd_row_stats: NULL argument");
        return SPD_ERR_INVALID_ARG;
    }
    if (n_reject_passes < 0 || n_reject_passes > 64 || (n_reject_passes > 0 && !(clip_sigma > 0.0f))) {
        set_error("spd_row_stats: need 0 <= n_reject_passes <= 64 and clip_sigma > 0 when rejecting (got %d, %g)",
                  n_reject_passes, static_cast<double>(clip_sigma));
        return SPD_ERR_INVALID_ARG;
    }
    return stats_run(plan, plane, clip_sigma, n_reject_passes, -1.0f, mean, sigma, nullptr,
                     static_cast<cudaStream_t>(cuda_stream));
}

int spd_row_stats_converge(const spd_plan* plan, const float* plane, float clip_sigma, int32_t max_reject_passes,
                           float rel_tol, float* mean, float* sigma, int32_t* n_passes, void* cuda_stream) {
    if (!plan || !plane || !mean || !sigma) {
        set_error("spd_row_stats_converge: NULL argument");
        return SPD_ERR_INVALID_ARG;
    }
    if (max_reject_passes < 1 || max_reject_passes > 64 || !(clip_sigma > 0.0f) || !(rel_tol >= 0.0f)) {
        set_error("spd_row_stats_converge: need 1 <= max_reject_passes <= 64, clip_sigma > 0, rel_tol >= 0 "
                  "(got %d, %g, %g)", max_reject_passes, static_cast<double>(clip_sigma), static_cast<double>(rel_tol));
        return SPD_ERR_INVALID_ARG;
    }
    return stats_run(plan, plane, clip_sigma, max_reject_passes, rel_tol, mean, sigma, n_passes,
                     static_cast<cudaStream_t>(cuda_stream));
}

int spd_cluster_candidates(const spd_plan* plan, const float* out_snr, const spd_candidate* list_in,
                           const int64_t* n_in, int64_t capacity_in, int32_t dm_radius, spd_candidate* list_out,
                           int64_t capacity_out, int64_t* n_out, void* cuda_stream) {
    if (!plan || !out_snr || !n_in || !n_out || capacity_in < 0 || capacity_out < 0 || dm_radius < 0 ||
        (capacity_in > 0 && !list_in) || (capacity_out > 0 && !list_out)) {
        set_error("spd_cluster_candidates: NULL argument, negative capacity or negative dm_radius");
        return SPD_ERR_INVALID_ARG;
    }
    return cluster_run(plan, out_snr, list_in, n_in, capacity_in, dm_radius, list_out, capacity_out, n_out,
                       static_cast<cudaStream_t>(cuda_stream));
}

int spd_run_host(spd_plan* plan, const float* plane, const float* mean, const float* sigma, float* out_snr,
                 void* out_width) {
    if (!plan || !plane || !mean || !sigma || !out_snr || !out_width) {
        set_error("spd_run_host: NULL argument");
        return SPD_ERR_INVALID_ARG;
    }
    int rc = prepare_host_staging(plan);
    if (rc != SPD_OK) return rc;
    HostStaging& h = plan->host;
    cudaError_t e;
    if ((e = cudaMemcpyAsync(h.d_mean, mean, sizeof(float) * plan->n_dm, cudaMemcpyHostToDevice, h.stream[0])) !=
            cudaSuccess ||
        (e = cudaMemcpyAsync(h.d_sigma, sigma, sizeof(float) * plan->n_dm, cudaMemcpyHostToDevice, h.stream[0])) !=
            cudaSuccess ||
        (e = cudaStreamSynchronize(h.stream[0])) != cudaSuccess)
        return cuda_fail(e, "copying mean / sigma to the device");
    // The workspace variant of the any-width-set path shares one workspace: one stream.
    const int n_streams = (runs_tree_kernel(plan) || plan->generic_tile > 0) ? 2 : 1;
    const size_t wb = static_cast<size_t>(plan->width_bytes);
    int64_t blk = 0;
    for (int64_t r0 = 0; r0 < plan->n_dm && rc == SPD_OK; r0 += h.rows_per_block, ++blk) {
        const int64_t rows = std::min<int64_t>(h.rows_per_block, plan->n_dm - r0);
        const int b = static_cast<int>(blk % 2);
        cudaStream_t st = h.stream[blk % n_streams];  // buffer b was last used two blocks ago on this stream
        const size_t off = static_cast<size_t>(r0) * static_cast<size_t>(plan->n_t);
        const size_t elems = static_cast<size_t>(rows) * static_cast<size_t>(plan->n_t);
        if ((e = cudaMemcpyAsync(h.d_plane[b], plane + off, elems * 4, cudaMemcpyHostToDevice, st)) != cudaSuccess) {
            rc = cuda_fail(e, "copying a row block to the device");
            break;
        }
        rc = run_rows(plan, rows, h.d_plane[b], h.d_mean + r0, h.d_sigma + r0, h.d_snr[b], h.d_width[b], 0.0f, nullptr,
                      st);
        if (rc != SPD_OK) break;
        if ((e = cudaMemcpyAsync(out_snr + off, h.d_snr[b], elems * 4, cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
            (e = cudaMemcpyAsync(static_cast<char*>(out_width) + off * wb, h.d_width[b], elems * wb,
                                 cudaMemcpyDeviceToHost, st)) != cudaSuccess)
            rc = cuda_fail(e, "copying results to the host");
    }
    // drain both streams whatever happened: no copy into the caller's buffers stays in flight
    for (int i = 0; i < 2; ++i)
        if ((e = cudaStreamSynchronize(h.stream[i])) != cudaSuccess && rc == SPD_OK)
            rc = cuda_fail(e, "waiting for the host run");
    return rc;
}

int spd_run_host_candidates(spd_plan* plan, const float* plane, const float* mean, const float* sigma,
                            float threshold, int32_t dm_radius, spd_candidate* list, int64_t capacity,
                            int64_t* n_found, int64_t* n_1d) {
    if (!plan || !plane || !mean || !sigma || !n_found || capacity < 0 || (capacity > 0 && !list)) {
        set_error("spd_run_host_candidates: NULL argument or negative capacity");
        return SPD_ERR_INVALID_ARG;
    }
    int rc = prepare_host_staging(plan);
    if (rc != SPD_OK) return rc;
    HostStaging& h = plan->host;
    cudaError_t e = cudaSuccess;
    const bool two_d = dm_radius >= 0;
    // device lists: the 1-D list of all blocks (at least 2^22 entries: a pulse gives hundreds of 1-D peaks),
    // the list after the 2-D stage (the caller's capacity)
    const int64_t cap1 = std::max<int64_t>(capacity, int64_t(1) << 22);
    const size_t act_bytes = activity_bytes_rows(plan, h.rows_per_block);
    for (int i = 0; i < 2 && e == cudaSuccess; ++i)
        if (!h.d_act[i]) e = cudaMalloc(&h.d_act[i], act_bytes);
    if (e == cudaSuccess && !h.d_counts) e = cudaMalloc(&h.d_counts, 2 * sizeof(int64_t));
    if (e == cudaSuccess && !h.h_counts) e = cudaMallocHost(&h.h_counts, 2 * sizeof(int64_t));
    if (e == cudaSuccess && h.list_cap < cap1) {
        cudaFree(h.d_list);
        h.d_list = nullptr;
        h.list_cap = 0;
        if ((e = cudaMalloc(&h.d_list, sizeof(spd_candidate) * static_cast<size_t>(cap1))) == cudaSuccess) h.list_cap = cap1;
    }
    if (e == cudaSuccess && two_d && h.list2_cap < std::max<int64_t>(capacity, 1)) {
        cudaFree(h.d_list2);
        h.d_list2 = nullptr;
        h.list2_cap = 0;
        const int64_t c2 = std::max<int64_t>(capacity, 1);
        if ((e = cudaMalloc(&h.d_list2, sizeof(spd_candidate) * static_cast<size_t>(c2))) == cudaSuccess) h.list2_cap = c2;
    }
    if (e == cudaSuccess && two_d && !h.d_snr_full)
        e = cudaMalloc(&h.d_snr_full, sizeof(float) * static_cast<size_t>(plan->n_dm) * static_cast<size_t>(plan->n_t));
    if (e != cudaSuccess) {
        set_error("allocating the candidate staging buffers failed: %s", cudaGetErrorString(e));
        cudaGetLastError();
        return SPD_ERR_ALLOC;
    }
    if ((e = cudaMemcpyAsync(h.d_mean, mean, sizeof(float) * plan->n_dm, cudaMemcpyHostToDevice, h.stream[0])) !=
            cudaSuccess ||
        (e = cudaMemcpyAsync(h.d_sigma, sigma, sizeof(float) * plan->n_dm, cudaMemcpyHostToDevice, h.stream[0])) !=
            cudaSuccess ||
        (e = cudaMemsetAsync(h.d_counts, 0, 2 * sizeof(int64_t), h.stream[0])) != cudaSuccess ||
        (e = cudaStreamSynchronize(h.stream[0])) != cudaSuccess)
        return cuda_fail(e, "copying mean / sigma to the device");
    const int n_streams = (runs_tree_kernel(plan) || plan->generic_tile > 0) ? 2 : 1;
    int64_t blk = 0;
    for (int64_t r0 = 0; r0 < plan->n_dm && rc == SPD_OK; r0 += h.rows_per_block, ++blk) {
        const int64_t rows = std::min<int64_t>(h.rows_per_block, plan->n_dm - r0);
        const int b = static_cast<int>(blk % 2);
        cudaStream_t st = h.stream[blk % n_streams];
        const size_t off = static_cast<size_t>(r0) * static_cast<size_t>(plan->n_t);
        const size_t elems = static_cast<size_t>(rows) * static_cast<size_t>(plan->n_t);
        if ((e = cudaMemcpyAsync(h.d_plane[b], plane + off, elems * 4, cudaMemcpyHostToDevice, st)) != cudaSuccess) {
            rc = cuda_fail(e, "copying a row block to the device");
            break;
        }
        float* const snr = two_d ? h.d_snr_full + off : h.d_snr[b];
        rc = run_rows(plan, rows, h.d_plane[b], h.d_mean + r0, h.d_sigma + r0, snr, h.d_width[b], threshold, h.d_act[b],
                      st);
        if (rc == SPD_OK)
            rc = candidates_run(plan, rows, r0, snr, h.d_width[b], h.d_act[b], threshold, h.d_list, h.list_cap,
                                h.d_counts, false, st);
    }
    for (int i = 0; i < 2; ++i)
        if ((e = cudaStreamSynchronize(h.stream[i])) != cudaSuccess && rc == SPD_OK)
            rc = cuda_fail(e, "waiting for the row blocks");
    if (rc != SPD_OK) return rc;
    cudaStream_t st = h.stream[0];
    if (two_d) {
        rc = cluster_run(plan, h.d_snr_full, h.d_list, h.d_counts, h.list_cap, dm_radius, h.d_list2, capacity,
                         h.d_counts + 1, st);
        if (rc != SPD_OK) return rc;
    }
    if ((e = cudaMemcpyAsync(h.h_counts, h.d_counts, 2 * sizeof(int64_t), cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
        (e = cudaStreamSynchronize(st)) != cudaSuccess)
        return cuda_fail(e, "reading the candidate counts");
    const int64_t found = two_d ? h.h_counts[1] : h.h_counts[0];
    const int64_t stored = std::min<int64_t>(found, two_d ? capacity : std::min<int64_t>(capacity, h.list_cap));
    if (stored > 0 &&
        ((e = cudaMemcpyAsync(list, two_d ? h.d_list2 : h.d_list, sizeof(spd_candidate) * static_cast<size_t>(stored),
                              cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
         (e = cudaStreamSynchronize(st)) != cudaSuccess))
        return cuda_fail(e, "copying the candidate list to the host");
    *n_found = found;
    if (n_1d) *n_1d = h.h_counts[0];
    return SPD_OK;
}

}  // extern "C"

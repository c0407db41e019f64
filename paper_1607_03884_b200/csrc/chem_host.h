// chem_host.h -- host-side definitions shared by the translation units of libchem.so (chem.cu, chem_tps.cu):
// the opaque mechanism object of include/chem.h, the error helper and the launch counter.
#pragma once
#include "../../include/chem.h"

#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>

#include "chem_common.cuh"

namespace chem_host {
int fail(int code, const char *fmt, ...);          // records the thread-local message of chem_last_error(), returns code
extern std::atomic<int64_t> g_launches;            // kernels launched by this library (chem_launch_count)
}  // namespace chem_host

#define CUDA_TRY(expr)                                                                                         \
    do {                                                                                                       \
        cudaError_t e_ = (expr);                                                                               \
        if (e_ != cudaSuccess) return chem_host::fail(CHEM_E_CUDA, "%s: %s", #expr, cudaGetErrorString(e_));   \
    } while (0)

struct chem_mech {
    chem::Tables t{};
    void *dev_blob = nullptr;   // one allocation holding every table
    int n_sm = 0;
    int max_smem_optin = 0;
    // algorithmic flop model
    double flops[5] = {0, 0, 0, 0, 0};
    double flops_t1[5] = {0, 0, 0, 0, 0};   // the same with 1 flop per transcendental instead of 20
    chem::FastTables fast{};    // exp-job tables of the warp-per-state and thread-per-state paths, if eligible
    void *fast_blob = nullptr;
    // host-buffer entry point: two streams for chunked copy/compute overlap (created on first use)
    cudaStream_t hs[2] = {nullptr, nullptr};
    int last_kernel = 0;        // kernel id of the last chem_integrate* launch (chem_last_kernel)
};

// Per-launch scratch (work-queue head, cost ordering, thread-per-state workspace) comes from the stream-ordered
// allocator (a memory pool of the library's own per device), so concurrent launches on different streams never share state.
namespace chem_host {
int scratch_alloc(void **p, size_t bytes, cudaStream_t st);
void scratch_free(void *p, cudaStream_t st);
int scratch_trim();
}  // namespace chem_host

// thread-per-state path (chem_tps.cu)
int chem_tps_available(const chem_mech *m);
int chem_tps_slots(const chem_mech *m);   // states in flight of one launch (lanes of all resident warps)
int chem_tps_launch(const chem_mech *m, int n, double P, const chem::RadauParams &prm, const double *y_in, double *y_out,
                    const chem_opts *o, chem_stats *stats, const int *order, cudaStream_t st);
// stiffness estimate per state for the start order (chem_opts.reorder = 2 / auto): keys[n] on the device, larger = costlier
int chem_tps_cost_keys(const chem_mech *m, int n, double P, const chem::RadauParams &prm, const double *y_in, const chem_opts *o,
                       int32_t *keys, cudaStream_t st);

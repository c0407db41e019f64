// chem_launch.inl -- host launch logic and the compute entry points of include/chem.h.
#include <cub/device/device_radix_sort.cuh>

namespace {

// group size: a warp per state up to 32 unknowns, a CTA per state above
inline int group_size(const chem_mech *m) { return m->t.n_sp <= 32 ? 32 : 128; }

template <typename K>
int configure(K kernel, const chem_mech *m, size_t smem, int *ctas_per_sm, int block = kBlock)
{
    if (smem > (size_t)m->max_smem_optin)
        return fail(CHEM_E_UNSUPPORTED, "mechanism needs %zu B of shared memory per CTA, device offers %d", smem, m->max_smem_optin);
    CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, block, smem));
    if (occ < 1) return fail(CHEM_E_UNSUPPORTED, "kernel does not fit on an SM");
    *ctas_per_sm = occ;
    return CHEM_OK;
}


// Optional cost ordering (chem_opts.reorder, "reordering IVPs to increase similarity"): with a work queue
// the order only decides WHEN a state starts; starting the expensive ones first shortens the tail of the launch.
__global__ void iota_kernel(int n, int *v)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) v[i] = i;
}
// Builds the start order in per-launch scratch (stream-ordered allocation; the caller frees *scratch after its launch).
int build_order(int n, const int32_t *cost, int **order_out, void **scratch, cudaStream_t st)
{
    size_t tmp_bytes = 0;
    cub::DeviceRadixSort::SortPairsDescending(nullptr, tmp_bytes, cost, (int32_t *)nullptr, (int *)nullptr, (int *)nullptr, n, 0, 32, st);
    const size_t head = ((size_t)3 * n * sizeof(int) + 255) & ~size_t(255);
    int rc = chem_host::scratch_alloc(scratch, head + tmp_bytes + 256, st);
    if (rc) return rc;
    int *idx = static_cast<int *>(*scratch), *ord = idx + n;
    int32_t *keys_out = reinterpret_cast<int32_t *>(ord + n);
    void *tmp = static_cast<char *>(*scratch) + head;
    iota_kernel<<<(n + 255) / 256, 256, 0, st>>>(n, idx);
    g_launches++;
    CUDA_TRY(cub::DeviceRadixSort::SortPairsDescending(tmp, tmp_bytes, cost, keys_out, idx, ord, n, 0, 32, st));
    g_launches += 3;   // cub: histogram + onesweep passes (not counted exactly)
    *order_out = ord;
    return CHEM_OK;
}

template <int G, bool JAC>
int launch_eval(const chem_mech *m, int n, double P, const double *y, double *out, cudaStream_t st)
{
    const size_t smem = work_doubles(m->t.n_sp, m->t.n_rx, G / 32, m->t.n_fo) * sizeof(double) * (block_of<G>() / G);
    int occ = 0;
    int rc = configure(eval_kernel<G, JAC>, m, smem, &occ, block_of<G>());
    if (rc) return rc;
    const int gpb = block_of<G>() / G;
    int grid = (n + gpb - 1) / gpb;
    if (grid > m->n_sm * occ) grid = m->n_sm * occ;
    eval_kernel<G, JAC><<<grid, block_of<G>(), smem, st>>>(m->t, n, P, y, out);
    g_launches++;
    CUDA_TRY(cudaGetLastError());
    return CHEM_OK;
}

// Every launch has its own work-queue head (4 bytes of stream-ordered scratch, zeroed on the stream), so launches on
// different streams with the same mechanism do not interfere.
template <int G>
int launch_integrate(const chem_mech *m, int n, double P, const RadauParams &prm, const double *y_in, double *y_out,
                     const chem_opts *o, chem_stats *stats, const int *order, cudaStream_t st)
{
    const size_t smem = work_doubles(m->t.n_sp, m->t.n_rx, G / 32, m->t.n_fo) * sizeof(double) * (block_of<G>() / G);
    int occ = 0;
    int rc = configure(integrate_kernel<G>, m, smem, &occ, block_of<G>());
    if (rc) return rc;
    const int gpb = block_of<G>() / G;
    int grid = (n + gpb - 1) / gpb;
    if (grid > m->n_sm * occ) grid = m->n_sm * occ;   // persistent: one wave, groups pull work from the queue
    void *scratch = nullptr;
    rc = chem_host::scratch_alloc(&scratch, 256, st);
    if (rc) return rc;
    int *counter = static_cast<int *>(scratch);
    cudaError_t e = cudaMemsetAsync(counter, 0, sizeof(int), st);
    if (e == cudaSuccess) {
        integrate_kernel<G><<<grid, block_of<G>(), smem, st>>>(m->t, n, P, o ? o->P_per_state : nullptr, prm, y_in, y_out, stats,
                                                        counter, order);
        g_launches++;
        e = cudaGetLastError();
    }
    chem_host::scratch_free(scratch, st);
    CUDA_TRY(e);
    return CHEM_OK;
}

int launch_integrate_warp(const chem_mech *m, int n, double P, const RadauParams &prm, const double *y_in, double *y_out,
                          const chem_opts *o, chem_stats *stats, const int *order, cudaStream_t st)
{
    const int wpb = kWarpBlock / 32;
    const size_t smem = ((size_t)m->fast.blob_doubles + (size_t)wpb * warp_ws_doubles(m->t.n_sp, m->t.n_rx)) * sizeof(double);
    if (smem > (size_t)m->max_smem_optin) return fail(CHEM_E_UNSUPPORTED, "warp kernel: shared memory");
    CUDA_TRY(cudaFuncSetAttribute(integrate_warp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, integrate_warp_kernel, kWarpBlock, smem));
    if (occ < 1) return fail(CHEM_E_UNSUPPORTED, "warp kernel does not fit on an SM");
    int grid = (n + wpb - 1) / wpb;
    if (grid > m->n_sm * occ) grid = m->n_sm * occ;   // persistent: one wave, warps pull states from the queue
    void *scratch = nullptr;
    const int rc = chem_host::scratch_alloc(&scratch, 256, st);
    if (rc) return rc;
    int *counter = static_cast<int *>(scratch);
    cudaError_t e = cudaMemsetAsync(counter, 0, sizeof(int), st);
    if (e == cudaSuccess) {
        integrate_warp_kernel<<<grid, kWarpBlock, smem, st>>>(m->t, m->fast, n, P, o ? o->P_per_state : nullptr, prm, y_in, y_out,
                                                              stats, counter, order);
        g_launches++;
        e = cudaGetLastError();
    }
    chem_host::scratch_free(scratch, st);
    CUDA_TRY(e);
    return CHEM_OK;
}

// eligible mechanism (chem_fast.inl) AND one CTA of kWarpBlock threads with its per-warp scratch fits in shared memory
// (N = 13: 218 KB; N = 16 does not fit: such mechanisms take the thread-per-state or the group kernel)
inline bool warp_path_available(const chem_mech *m)
{
    if (!m->fast.enabled) return false;
    const size_t smem = ((size_t)m->fast.blob_doubles + (size_t)(kWarpBlock / 32) * warp_ws_doubles(m->t.n_sp, m->t.n_rx)) * sizeof(double);
    return smem <= (size_t)m->max_smem_optin;
}

}  // namespace

extern "C" int chem_rhs(const chem_mech *m, int32_t n, double P, const double *y, double *f, void *stream)
{
    if (!m || n < 0 || (n > 0 && (!y || !f))) return fail(CHEM_E_ARG, "bad argument");
    if (n == 0) return CHEM_OK;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    return group_size(m) == 32 ? launch_eval<32, false>(m, n, P, y, f, st) : launch_eval<128, false>(m, n, P, y, f, st);
}

extern "C" int chem_jacobian(const chem_mech *m, int32_t n, double P, const double *y, double *J, void *stream)
{
    if (!m || n < 0 || (n > 0 && (!y || !J))) return fail(CHEM_E_ARG, "bad argument");
    if (n == 0) return CHEM_OK;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    return group_size(m) == 32 ? launch_eval<32, true>(m, n, P, y, J, st) : launch_eval<128, true>(m, n, P, y, J, st);
}

extern "C" int chem_lu_solve(int32_t n, int32_t batch, int32_t is_complex, const double *A, const double *b, double *x,
                             int32_t *info, void *stream)
{
    if (n < 1 || batch < 0 || (batch > 0 && (!A || !b || !x))) return fail(CHEM_E_ARG, "bad argument");
    if (batch == 0) return CHEM_OK;
    if (n <= 16) {   // the warp path's routines (Gauss-Jordan inverse + matrix-vector solve)
        const size_t sm = ((size_t)2 * n * (n | 1) + 34) * sizeof(double2);
        const int g = batch < 65535 ? batch : 65535;
        lu_solve_warp_kernel<<<g, 32, sm, static_cast<cudaStream_t>(stream)>>>(n, batch, is_complex, A, b, x, info);
        g_launches++;
        CUDA_TRY(cudaGetLastError());
        return CHEM_OK;
    }
    if (n <= 64) {   // the group kernels' routines (fused real + complex LU, pivot-ordered factors, chain-free solves)
        const size_t sm = ((size_t)3 * n * (n + 1) + 6 * n) * sizeof(double) + (size_t)4 * n * sizeof(int) + 16;
        CUDA_TRY(cudaFuncSetAttribute(lu2_solve_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
        const int g = batch < 65535 ? batch : 65535;
        lu2_solve_kernel<<<g, 128, sm, static_cast<cudaStream_t>(stream)>>>(n, batch, is_complex, A, b, x, info);
        g_launches++;
        CUDA_TRY(cudaGetLastError());
        return CHEM_OK;
    }
    const size_t smem = ((size_t)2 * n * n + 2 * n) * sizeof(double) + (size_t)n * sizeof(int) + 16;
    int dev = 0, optin = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    if (smem > (size_t)optin) return fail(CHEM_E_UNSUPPORTED, "n = %d does not fit in shared memory", n);
    CUDA_TRY(cudaFuncSetAttribute(lu_solve_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int grid = batch < 65535 ? batch : 65535;
    lu_solve_kernel<<<grid, 32, smem, static_cast<cudaStream_t>(stream)>>>(n, batch, is_complex, A, b, x, info);
    g_launches++;
    CUDA_TRY(cudaGetLastError());
    return CHEM_OK;
}

namespace {
// Kernel ids (chem_opts.kernel, chem_last_kernel): 1 shared-memory group kernel, 2 warp-per-state, 3 thread-per-state.
// Auto picks the fastest measured mapping (profiles/r2_mapping_config1.md, r2_mapping_config2.md, r3_tail_config1.md): for an
// eligible small mechanism the thread-per-state kernel when the batch fills its lanes at least six times over -- with the
// ordered start it takes 11.7 ms for 262,144 states at dt = 1e-6 s against 14.5 ms for the warp-per-state kernel, 10.0 against
// 3.7 ms for 65,536: break-even near 200,000 states (it was 300,000 without the ordering) -- else the warp-per-state
// kernel; the group kernel for everything else.
int pick_kernel(const chem_mech *m, int n, const chem_opts *o)
{
    const int want = o ? o->kernel : 0;
    if (want != 0) return want;
    if (chem_tps_available(m) && (long long)n >= 6LL * chem_tps_slots(m)) return 3;
    if (warp_path_available(m)) return 2;
    return 1;
}

int integrate_impl(const chem_mech *m, int32_t n, double P, double t_end, double rtol, double atol, const double *y_in,
                   double *y_out, const chem_opts *o, chem_stats *stats, cudaStream_t st)
{
    if (!m || n < 0 || (n > 0 && (!y_in || !y_out))) return fail(CHEM_E_ARG, "bad argument");
    if (!(t_end > 0.0) || !(rtol > 0.0) || !(atol > 0.0)) return fail(CHEM_E_ARG, "t_end, rtol and atol must be positive");
    if (o && (o->kernel < 0 || o->kernel > 3)) return fail(CHEM_E_ARG, "chem_opts.kernel must be 0..3");
    if (n == 0) return CHEM_OK;
    RadauParams prm;
    prm.t_end = t_end; prm.rtol = rtol; prm.atol = atol;
    prm.h0 = o ? o->h0 : 0.0;
    prm.max_steps = o ? o->max_steps : 0;
    prm.newton_max = o ? o->newton_max : 0;
    prm.fd_jacobian = o ? o->fd_jacobian : 0;
    prm.fixed_steps = o ? o->fixed_steps : 0;
    prm.rtol_t = 0.1 * std::pow(rtol, 2.0 / 3.0);
    prm.atol_t = prm.rtol_t * (atol / rtol);
    prm.fnewt = std::fmax(10.0 * 2.220446049250313e-16 / prm.rtol_t, std::fmin(0.03, std::sqrt(prm.rtol_t)));
    prm.inv_fnewt = 1.0 / prm.fnewt; prm.inv_n = 1.0 / m->t.n_sp; prm.inv_3n = 1.0 / (3 * m->t.n_sp);
    const int kernel = pick_kernel(m, n, o);
    if (kernel == 2 && !warp_path_available(m)) return fail(CHEM_E_UNSUPPORTED, "warp-per-state kernel not available for this mechanism");
    if (kernel == 3 && !chem_tps_available(m)) return fail(CHEM_E_UNSUPPORTED, "thread-per-state kernel not available for this mechanism");
    int *order = nullptr;
    void *order_scratch = nullptr, *key_scratch = nullptr;
    // Start order (chem_opts.reorder): 1 = by the caller's cost_hint; 2 = by the library's own stiffness estimate
    // (chem_tps_cost_keys: one source term per state + a radix sort, 1.8 ms per million h2co-shaped states); 0 = auto: the
    // estimate where it is measured to pay (profiles/r3_tail_config1.md): the thread-per-state kernel from four times its
    // lanes on (its launch otherwise ends with a few long states and idle lanes: 40.2 -> 34.9 ms on config 1) and the
    // warp-per-state kernel from four waves of its warps on (16,384 states: 1.49 -> 1.22 ms; at 4,096 states the extra
    // launches cost more than the order gives); < 0 = off.  Bits of the results never depend on it.
    const int reorder = o ? o->reorder : 0;
    bool auto_order = false;
    if (reorder == 0 && chem_tps_available(m)) {
        if (kernel == 3) auto_order = (long long)n >= 4LL * chem_tps_slots(m);
        else if (kernel == 2) auto_order = (long long)n >= 4LL * m->n_sm * (kWarpBlock / 32);
    }
    if (reorder < -1 || reorder > 2) return fail(CHEM_E_ARG, "chem_opts.reorder must be -1..2");
    if (reorder == 1 && o->cost_hint) {
        const int rc = build_order(n, o->cost_hint, &order, &order_scratch, st);
        if (rc) { chem_host::scratch_free(order_scratch, st); return rc; }
    } else if (reorder == 2 || auto_order) {
        int rc = chem_host::scratch_alloc(&key_scratch, (size_t)n * sizeof(int32_t), st);
        if (rc == CHEM_OK) rc = chem_tps_cost_keys(m, n, P, prm, y_in, o, static_cast<int32_t *>(key_scratch), st);
        if (rc == CHEM_OK) rc = build_order(n, static_cast<const int32_t *>(key_scratch), &order, &order_scratch, st);
        if (rc) { chem_host::scratch_free(order_scratch, st); chem_host::scratch_free(key_scratch, st); return rc; }
    }
    int rc;
    if (kernel == 3) rc = chem_tps_launch(m, n, P, prm, y_in, y_out, o, stats, order, st);
    else if (kernel == 2) rc = launch_integrate_warp(m, n, P, prm, y_in, y_out, o, stats, order, st);
    else rc = group_size(m) == 32 ? launch_integrate<32>(m, n, P, prm, y_in, y_out, o, stats, order, st)
                                  : launch_integrate<128>(m, n, P, prm, y_in, y_out, o, stats, order, st);
    chem_host::scratch_free(order_scratch, st);
    chem_host::scratch_free(key_scratch, st);
    if (rc == CHEM_OK) const_cast<chem_mech *>(m)->last_kernel = kernel;
    return rc;
}
}  // namespace

extern "C" int chem_last_kernel(const chem_mech *m) { return m ? m->last_kernel : 0; }

extern "C" int chem_integrate_ex(const chem_mech *m, int32_t n, double P, double t_end, double rtol, double atol,
                                 const double *y_in, double *y_out, const chem_opts *o, chem_stats *stats, void *stream)
{
    return integrate_impl(m, n, P, t_end, rtol, atol, y_in, y_out, o, stats, static_cast<cudaStream_t>(stream));
}

extern "C" int chem_integrate(const chem_mech *m, int32_t n, double P, double t_end, double rtol, double atol,
                              const double *y_in, double *y_out, void *stream)
{
    return chem_integrate_ex(m, n, P, t_end, rtol, atol, y_in, y_out, nullptr, nullptr, stream);
}

extern "C" int chem_integrate_host(const chem_mech *m, int32_t n, double P, double t_end, double rtol, double atol,
                                   const double *y_in_host, double *y_out_host, const chem_opts *o, chem_stats *stats_host)
{
    if (!m || n < 0 || (n > 0 && (!y_in_host || !y_out_host))) return fail(CHEM_E_ARG, "bad argument");
    if (n == 0) return CHEM_OK;
    chem_mech *mm = const_cast<chem_mech *>(m);
    const int N = m->t.n_sp;
    const size_t ybytes = (size_t)n * N * sizeof(double), sbytes = stats_host ? (size_t)n * sizeof(chem_stats) : 0;
    constexpr int kStreams = 2;
    for (int i = 0; i < kStreams; i++)
        if (!mm->hs[i]) CUDA_TRY(cudaStreamCreateWithFlags(&mm->hs[i], cudaStreamNonBlocking));
    // Page-locked host buffers are mapped into the device's address space (unified addressing): the kernel then reads
    // each state from host memory when it starts it and writes the result back when it finishes it, so the transfers
    // ride inside the one persistent launch instead of before and after it (measured on B200 / PCIe Gen5, config 1: 59.1 ms
    // device-resident, 60.8 ms through mapped pinned buffers; staged copies of the 2 x 109 MB cost 2.0 + 2.5 ms more,
    // and chunking them over streams does not hide them because consecutive persistent launches do not overlap).
    {
        auto mapped = [](const void *h) -> void * {
            cudaPointerAttributes at;
            if (cudaPointerGetAttributes(&at, h) != cudaSuccess) { cudaGetLastError(); return nullptr; }
            return at.type == cudaMemoryTypeHost ? at.devicePointer : nullptr;
        };
        void *din = mapped(y_in_host), *dout = mapped(y_out_host), *dst = stats_host ? mapped(stats_host) : nullptr;
        if (din && dout && (!stats_host || dst)) {
            chem_opts oc{};
            if (o) oc = *o;
            // caller's cost hints are not used here; auto stays auto: the estimate kernel then reads the input once more
            // through the mapping (2 ms per 109 MB over PCIe Gen5), which the ordered launch more than pays back
            oc.reorder = o && o->reorder < 0 ? -1 : 0;
            oc.cost_hint = nullptr;
            const int rc0 = integrate_impl(m, n, P, t_end, rtol, atol, static_cast<const double *>(din), static_cast<double *>(dout),
                                           &oc, static_cast<chem_stats *>(dst), mm->hs[0]);
            if (rc0 != CHEM_OK) return rc0;
            CUDA_TRY(cudaStreamSynchronize(mm->hs[0]));
            return CHEM_OK;
        }
    }
    // pageable host memory: staged copies, two chunks on two streams
    void *buf = nullptr;
    int rc = chem_host::scratch_alloc(&buf, ybytes + sbytes + 256, mm->hs[0]);
    if (rc) return rc;
    {                                                   // the block is used from both streams
        const cudaError_t es = cudaStreamSynchronize(mm->hs[0]);
        if (es != cudaSuccess) {
            chem_host::scratch_free(buf, mm->hs[0]);
            return fail(CHEM_E_CUDA, "chem_integrate_host: %s", cudaGetErrorString(es));
        }
    }
    double *d_y = static_cast<double *>(buf);
    chem_stats *d_st = stats_host ? reinterpret_cast<chem_stats *>(static_cast<char *>(buf) + ((ybytes + 255) & ~size_t(255))) : nullptr;
    const int n_chunks = n >= 65536 ? 2 : 1;
    // the kernel is chosen once, from the whole batch: a chunk must not fall back to another mapping (and other bits)
    // just because it is half as long (pick_kernel depends on n)
    const int kernel_all = pick_kernel(m, n, o);
    cudaError_t e = cudaSuccess;
    for (int c = 0; c < n_chunks && rc == CHEM_OK && e == cudaSuccess; c++) {
        const int lo = (int)((long long)n * c / n_chunks), hi = (int)((long long)n * (c + 1) / n_chunks);
        if (hi == lo) continue;
        cudaStream_t st = mm->hs[c % kStreams];
        chem_opts oc{};
        if (o) {
            oc = *o;
            if (oc.P_per_state) oc.P_per_state += lo;
        }
        oc.reorder = o && o->reorder < 0 ? -1 : 0;   // caller's cost hints are device arrays of the whole batch: not used; auto per chunk
        oc.cost_hint = nullptr;
        oc.kernel = kernel_all;
        const size_t off = (size_t)lo * N, cnt = (size_t)(hi - lo) * N;
        e = cudaMemcpyAsync(d_y + off, y_in_host + off, cnt * sizeof(double), cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) break;
        rc = integrate_impl(m, hi - lo, P, t_end, rtol, atol, d_y + off, d_y + off, &oc, d_st ? d_st + lo : nullptr, st);
        if (rc != CHEM_OK) break;
        e = cudaMemcpyAsync(y_out_host + off, d_y + off, cnt * sizeof(double), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && stats_host)
            e = cudaMemcpyAsync(stats_host + lo, d_st + lo, (size_t)(hi - lo) * sizeof(chem_stats), cudaMemcpyDeviceToHost, st);
    }
    for (int i = 0; i < kStreams; i++) {
        const cudaError_t e2 = cudaStreamSynchronize(mm->hs[i]);
        if (e == cudaSuccess) e = e2;
    }
    chem_host::scratch_free(buf, mm->hs[0]);
    if (rc != CHEM_OK) return rc;
    if (e != cudaSuccess) return fail(CHEM_E_CUDA, "chem_integrate_host: %s", cudaGetErrorString(e));
    return CHEM_OK;
}

// ------------------------------------------------------------------------------------------------ fp64 peak probe
// Dependent-free DFMA streams (8 accumulators per thread, full occupancy): measures the fp64 FMA rate that the "alu"
// roofline of DESIGN.md 7 is derived from (148 SM x 64 lanes x 2 flop x clock).  Diagnostic only, not on the hot path.
namespace {
__global__ void __launch_bounds__(256) fp64_probe_kernel(int iters, double seed, double *sink)
{
    double a0 = seed + threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double m = 1.0 - 1e-9, c = 1e-9;
#pragma unroll 4
    for (int i = 0; i < iters; i++) {
        a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
        a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
    const double r = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (r == 12345.678) sink[0] = r;      // never true: keeps the loop alive
}
}  // namespace

extern "C" int chem_fp64_probe(int32_t iters, int32_t reps, double *tflops_best)
{
    if (iters < 1 || reps < 1 || !tflops_best) return fail(CHEM_E_ARG, "bad argument");
    int dev = 0, n_sm = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    double *sink = nullptr;
    CUDA_TRY(cudaMalloc(&sink, 8));
    cudaEvent_t e0, e1;
    CUDA_TRY(cudaEventCreate(&e0));
    CUDA_TRY(cudaEventCreate(&e1));
    const int grid = n_sm * 8;
    double best = 0.0;
    for (int r = 0; r < reps + 1; r++) {
        cudaEventRecord(e0);
        fp64_probe_kernel<<<grid, 256>>>(iters, 1.0, sink);
        cudaEventRecord(e1);
        g_launches++;
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { cudaFree(sink); return fail(CHEM_E_CUDA, "fp64 probe: %s", cudaGetErrorString(e)); }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double tf = (double)grid * 256 * 8 * 2.0 * iters / (ms * 1e-3) / 1e12;
        if (r > 0 && tf > best) best = tf;       // the first launch is a warm-up
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
    *tflops_best = best;
    return CHEM_OK;
}

// chem_tps.cu -- thread-per-state integrator: launcher, the instantiations for runtime N and N = 13, and the test hook of
// its linear algebra.  The kernel itself is in chem_tps_kernel.cuh, the device routines in chem_tps.cuh.
#include "chem_tps_kernel.cuh"

#include <cstdlib>

using namespace chem;
using namespace chem::tps;

CHEM_TPS_INSTANTIATE(0)
CHEM_TPS_INSTANTIATE(13)

namespace {

size_t tps_smem(const chem_mech *m, int warps)
{
    const Lay L = make_lay(m->t.n_sp, m->t.n_rx);
    return ((size_t)((m->fast.blob_doubles + 31) & ~31) + (size_t)warps * L.n_sm * 32) * sizeof(double);
}
// warps out of every 8 whose LU factors stay resident in L2 (chem_tps.cuh, l2_policy); CHEM_TPS_L2_KEEP overrides the
// default for experiments (0..8)
int tps_l2_keep()
{
    static const int v = [] {
        const char *e = std::getenv("CHEM_TPS_L2_KEEP");
        const int k = e ? std::atoi(e) : 8;      // measured (profiles/r3_tps_config1.md): all factors evict_last is the fastest
        return k < 0 ? 0 : (k > 8 ? 8 : k);
    }();
    return v;
}
int tps_warps(const chem_mech *m)
{
    (void)m;
    return 4;          // two CTAs of four warps per SM (or one, if shared memory holds only one); two CTAs of three warps, so
                       // that the factors of all resident lanes fit in L2 (115 MB), is 22 % SLOWER (profiles/r3_tps_config1.md)
}

}  // namespace

int chem_tps_available(const chem_mech *m)
{
    if (!m->fast.enabled) return 0;
    return tps_smem(m, 4) <= (size_t)m->max_smem_optin;
}

int chem_tps_slots(const chem_mech *m) { return m->n_sm * 32 * 8; }

int chem_tps_launch(const chem_mech *m, int n, double P, const RadauParams &prm, const double *y_in, double *y_out,
                    const chem_opts *o, chem_stats *stats, const int *order, cudaStream_t st)
{
    using chem_host::fail;
    if (!chem_tps_available(m)) return fail(CHEM_E_UNSUPPORTED, "thread-per-state kernel not available for this mechanism");
    const Lay L = make_lay(m->t.n_sp, m->t.n_rx);
    const int warps = tps_warps(m);
    const size_t smem = tps_smem(m, warps);
    int grid = (n + 32 * warps - 1) / (32 * warps);
    if (grid > m->n_sm * (8 / warps)) grid = m->n_sm * (8 / warps);   // persistent: 8 warps per SM, lanes pull states from the queue
    const size_t ws_bytes = (size_t)grid * warps * L.n_gw * 32 * sizeof(double);
    void *scratch = nullptr;
    int rc = chem_host::scratch_alloc(&scratch, ws_bytes + 256, st);
    if (rc) return rc;
    TpsArgs a;
    a.n_states = n; a.N = L.N; a.NR = L.NR; a.n_sm = L.n_sm; a.n_gw = L.n_gw;
    a.P = P; a.tmid = m->fast.tmid;
    a.P_per_state = o ? o->P_per_state : nullptr;
    a.prm = prm;
    a.y_in = y_in; a.y_out = y_out; a.stats = stats;
    a.counter = reinterpret_cast<int *>(static_cast<char *>(scratch) + ws_bytes);
    a.order = order;
    a.gws = static_cast<double *>(scratch);
    a.blob = m->fast.blob; a.blob_doubles = m->fast.blob_doubles;
    a.l2_keep = tps_l2_keep();
    cudaError_t e = cudaMemsetAsync(a.counter, 0, sizeof(int), st);
    if (e == cudaSuccess) {
        // compile-time-N instantiations for 8 <= N <= 16, runtime-N routines below that
        typedef cudaError_t (*launch_fn)(const TpsArgs &, int, size_t, cudaStream_t);
        static const launch_fn table[17] = {chem_tps_launch_nt0, chem_tps_launch_nt0, chem_tps_launch_nt0, chem_tps_launch_nt0,
                                            chem_tps_launch_nt0, chem_tps_launch_nt0, chem_tps_launch_nt0, chem_tps_launch_nt0,
                                            chem_tps_launch_nt8, chem_tps_launch_nt9, chem_tps_launch_nt10, chem_tps_launch_nt11,
                                            chem_tps_launch_nt12, chem_tps_launch_nt13, chem_tps_launch_nt14, chem_tps_launch_nt15,
                                            chem_tps_launch_nt16};
        e = table[L.N](a, grid, smem, st);
        chem_host::g_launches++;
    }
    chem_host::scratch_free(scratch, st);
    if (e != cudaSuccess) return fail(CHEM_E_CUDA, "thread-per-state launch: %s", cudaGetErrorString(e));
    return CHEM_OK;
}

// ------------------------------------------------------------------------------------------------ stiffness estimate
// Cost estimate for the start order of a launch (chem_opts.reorder = 2 / auto; "reordering IVPs to increase
// similarity of stiffness"; L184: a warp waits for its most expensive thread).  With a work queue the order of the states
// only decides WHEN each one starts; started in order of decreasing cost, the long ones do not end up alone at the end of
// the launch with every other lane idle.  The estimate is the quantity the controller itself would look at first:
// key = 16 log2(1 + t_end || f(y0) / (atol + rtol |y0|) ||_rms), i.e. how many tolerances the state moves over the global
// step at its initial rate, in sixteenths of an octave, 0..1023.  Measured on B200 (profiles/r3_tail_config1.md): ordering by
// it recovers 90 % of what ordering by the true step counts of a previous run gives.  One source term per state, thread
// per state, states loaded as coalesced rows exactly as the integration kernel loads them.
namespace {
__global__ void __launch_bounds__(128) tps_cost_kernel(const __grid_constant__ TpsArgs a, int32_t *key)
{
    extern __shared__ double smem[];
    for (int i = threadIdx.x; i < a.blob_doubles; i += 128) smem[i] = a.blob[i];
    __syncthreads();
    const double *tab = smem;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int N = a.N, NR = a.NR;
    double *sm = smem + ((a.blob_doubles + 31) & ~31) + (size_t)wib * a.n_sm * 32 + lane;
    double *wsm = sm - lane, *y = sm, *f = sm + oZ(N) * 32;
    const double rtol = a.prm.rtol, atol = a.prm.atol, t_end = a.prm.t_end, invN = a.prm.inv_n;
    for (long long base = ((long long)blockIdx.x * 4 + wib) * 32; base < a.n_states; base += (long long)gridDim.x * 128) {
        if (base + 32 <= a.n_states) {                 // full tile: the 32 row loads are independent, keep them in flight together
#pragma unroll 8
            for (int l = 0; l < 32; l++)
                if (lane < N) wsm[lane * 32 + l] = a.y_in[(size_t)(base + l) * N + lane];
        } else {
            for (int l = 0; l < 32 && base + l < a.n_states; l++)
                if (lane < N) wsm[lane * 32 + l] = a.y_in[(size_t)(base + l) * N + lane];
        }
        __syncwarp();
        const long long s = base + lane;
        if (s < a.n_states) {
            const double P = a.P_per_state ? a.P_per_state[s] : a.P;
            rhs(tab, sm, N, NR, a.tmid, P, rcp_f(P), y, 0.0, f);
            double e = 0.0;
#pragma unroll 1
            for (int i = 0; i < N; i++) { const double r = TL(f, i) / (atol + rtol * fabs(TL(y, i))); e = fma(r, r, e); }
            const double k = 16.0 * log2(1.0 + t_end * sqrt(e * invN));
            key[s] = k >= 1023.0 ? 1023 : (k > 0.0 ? (int32_t)k : 0);          // NaN (non-finite state) -> 0
        }
        __syncwarp();
    }
}
}  // namespace

int chem_tps_cost_keys(const chem_mech *m, int n, double P, const RadauParams &prm, const double *y_in, const chem_opts *o,
                       int32_t *keys, cudaStream_t st)
{
    using chem_host::fail;
    if (!chem_tps_available(m)) return fail(CHEM_E_UNSUPPORTED, "the stiffness estimate (reorder = 2) needs a small mechanism (thread-per-state source term)");
    const Lay L = make_lay(m->t.n_sp, m->t.n_rx);
    const size_t smem = tps_smem(m, 4);
    CUDA_TRY(cudaFuncSetAttribute(tps_cost_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, tps_cost_kernel, 128, smem));
    if (occ < 1) return fail(CHEM_E_UNSUPPORTED, "stiffness-estimate kernel does not fit on an SM");
    int grid = (n + 127) / 128;
    if (grid > m->n_sm * occ) grid = m->n_sm * occ;
    TpsArgs a{};
    a.n_states = n; a.N = L.N; a.NR = L.NR; a.n_sm = L.n_sm; a.n_gw = L.n_gw;
    a.P = P; a.tmid = m->fast.tmid;
    a.P_per_state = o ? o->P_per_state : nullptr;
    a.prm = prm;
    a.y_in = y_in;
    a.blob = m->fast.blob; a.blob_doubles = m->fast.blob_doubles;
    tps_cost_kernel<<<grid, 128, smem, st>>>(a, keys);
    chem_host::g_launches++;
    CUDA_TRY(cudaGetLastError());
    return CHEM_OK;
}

// ------------------------------------------------------------------------------------------------ test hook
// The linear algebra of one Radau step exactly as the integration kernel runs it (chem_tps.cuh: lu_pair_t<N> / solve3_t<N>
// for 8 <= N <= 16, the runtime-N lu_pair / solve3 below that -- the same table as chem_tps_launch), one system per lane:
// (fac1 I - J) x1 = b1  and  ((alphn + i betan) I - J)(x2 + i x3) = b2 + i b3.  The kernel is tps_solve_kernel<NT> in
// chem_tps_kernel.cuh, instantiated beside the integration kernel of the same N.
extern "C" int chem_tps_radau_solve(int32_t n, int32_t batch, const double *J, double fac1, double alphn, double betan,
                                    const double *b, double *x, int32_t *info, void *stream)
{
    using chem_host::fail;
    if (n < 1 || n > 16 || batch < 0 || (batch > 0 && (!J || !b || !x))) return fail(CHEM_E_ARG, "bad argument (1 <= n <= 16)");
    if (batch == 0) return CHEM_OK;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int grid = (batch + 127) / 128;
    const size_t smem = (size_t)4 * 6 * n * 32 * sizeof(double);
    void *ws = nullptr;
    const int rc = chem_host::scratch_alloc(&ws, (size_t)grid * 4 * 4 * n * n * 32 * sizeof(double), st);
    if (rc) return rc;
    typedef cudaError_t (*solve_fn)(int, int, const double *, double, double, double, const double *, double *, int *, double *, int,
                                    size_t, cudaStream_t);
    static const solve_fn table[17] = {chem_tps_solve_nt0, chem_tps_solve_nt0, chem_tps_solve_nt0, chem_tps_solve_nt0,
                                       chem_tps_solve_nt0, chem_tps_solve_nt0, chem_tps_solve_nt0, chem_tps_solve_nt0,
                                       chem_tps_solve_nt8, chem_tps_solve_nt9, chem_tps_solve_nt10, chem_tps_solve_nt11,
                                       chem_tps_solve_nt12, chem_tps_solve_nt13, chem_tps_solve_nt14, chem_tps_solve_nt15,
                                       chem_tps_solve_nt16};
    cudaError_t e = table[n](n, batch, J, fac1, alphn, betan, b, x, info, static_cast<double *>(ws), grid, smem, st);
    if (e == cudaSuccess) { chem_host::g_launches++; e = cudaGetLastError(); }
    chem_host::scratch_free(ws, st);
    if (e != cudaSuccess) return fail(CHEM_E_CUDA, "chem_tps_radau_solve: %s", cudaGetErrorString(e));
    return CHEM_OK;
}

// chem_kernels.inl -- kernels and launch logic; included at the end of chem.cu.

namespace {

constexpr int kBlock = 128;   // threads per CTA of the warp-group kernels (G = 32); a CTA-group kernel has G threads
template <int G>
__host__ __device__ constexpr int block_of() { return G > kBlock ? G : kBlock; }

// Group <-> CTA mapping: G == 32 -> four warp-groups per CTA, G >= 128 -> the CTA is the group.
template <int G>
__device__ __forceinline__ int group_in_block() { return G == 32 ? (int)(threadIdx.x >> 5) : 0; }

// Next state index from the work queue (PAPER.md L194 names load imbalance between IVPs; groups that
// finish early pull new states).  Uniform across the group.
template <int G>
__device__ __forceinline__ int next_state(int *counter, int *bcast)
{
    int s = 0;
    if (G == 32) {
        if ((threadIdx.x & 31) == 0) s = atomicAdd(counter, 1);
        s = __shfl_sync(0xffffffffu, s, 0);
    } else {
        __syncthreads();
        if (threadIdx.x == 0) *bcast = atomicAdd(counter, 1);
        __syncthreads();
        s = *bcast;
    }
    return s;
}

template <int G>
__global__ void __launch_bounds__(block_of<G>(), G > kBlock ? 2 : 1) integrate_kernel(Tables t_arg, int n_states, double P, const double *P_per_state,
                                                           RadauParams prm, const double *y_in,
                                                           double *y_out, chem_stats *stats, int *counter,
                                                           const int *order)
{
    extern __shared__ double smem[];
    __shared__ int bcast;
    // the table descriptor in (static) shared memory: the out-of-line routines take it by reference, and a reference to
    // the kernel parameter would be a local-memory copy (40,000 local loads per GRI state, 45 % of them L1 misses)
    __shared__ Tables t;
    if (threadIdx.x == 0) t = t_arg;
    __syncthreads();
    const int N = t.n_sp, NR = t.n_rx;
    const size_t wd = work_doubles(N, NR, Grp<G>::NW, t.n_fo);
    Work w = carve(smem + (size_t)group_in_block<G>() * wd, N, NR, Grp<G>::NW, t.n_fo);
    const int lane = Grp<G>::lane();
    for (;;) {
        const int q = next_state<G>(counter, &bcast);
        if (q >= n_states) break;
        const int s = order ? order[q] : q;
        for (int i = lane; i < N; i += G) w.y[i] = y_in[(size_t)s * N + i];
        Grp<G>::sync();
        RadauResult r;
        radau_state<G>(t, w, P_per_state ? P_per_state[s] : P, prm, r);
        Grp<G>::sync();
        for (int i = lane; i < N; i += G) y_out[(size_t)s * N + i] = w.y[i];
        if (stats && lane == 0) {
            chem_stats o;
            o.status = r.status; o.nstep = r.nstep; o.naccpt = r.naccpt; o.nrejct = r.nrejct; o.nfcn = r.nfcn;
            o.njac = r.njac; o.ndec = r.ndec; o.nsol = r.nsol; o.nnewt_fail = r.nnewt_fail; o.reserved = 0;
            o.h_last = r.h_last;
            stats[s] = o;
        }
        Grp<G>::sync();
    }
}

// Compact warp-per-state integrator (chem_warp.cuh / chem_radau_warp.cuh): 8 warps per CTA.
constexpr int kWarpBlock = 640;

__global__ void __launch_bounds__(kWarpBlock, 1) integrate_warp_kernel(Tables t, FastTables ft, int n_states, double P,
                                                                    const double *P_per_state, RadauParams prm,
                                                                    const double *y_in, double *y_out,
                                                                    chem_stats *stats, int *counter, const int *order)
{
    extern __shared__ double smem[];
    for (int i = threadIdx.x; i < ft.blob_doubles; i += kWarpBlock) smem[i] = ft.blob[i];   // stage the tables once per CTA
    __syncthreads();
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int N = t.n_sp;
    double *ws = smem + ft.blob_doubles + (size_t)wib * warp_ws_doubles(N, t.n_rx);
    if (lane >= N) { ws[kWsC + lane] = 1.0; ws[kWsC + 32 + lane] = 1.0; ws[kWsC + 64 + lane] = 1.0; }   // C[s][31] = 1: unity factor
    __syncwarp();
    for (;;) {
        int q = 0;
        if (lane == 0) q = atomicAdd(counter, 1);
        q = __shfl_sync(0xffffffffu, q, 0);
        if (q >= n_states) break;
        if (order) q = order[q];
        double y = lane < N ? y_in[(size_t)q * N + lane] : 0.0;
        RadauResult r;
        radau_state_warp(t, smem, ws, ft.tmid, P_per_state ? P_per_state[q] : P, prm, y, r);
        if (lane < N) y_out[(size_t)q * N + lane] = y;
        if (stats && lane == 0) {
            chem_stats o;
            o.status = r.status; o.nstep = r.nstep; o.naccpt = r.naccpt; o.nrejct = r.nrejct; o.nfcn = r.nfcn;
            o.njac = r.njac; o.ndec = r.ndec; o.nsol = r.nsol; o.nnewt_fail = r.nnewt_fail; o.reserved = 0;
            o.h_last = r.h_last;
            stats[q] = o;
        }
        __syncwarp();
    }
}

// Source term / Jacobian for a batch (static round-robin over groups).
template <int G, bool JAC>
__global__ void __launch_bounds__(block_of<G>()) eval_kernel(Tables t_arg, int n_states, double P, const double *__restrict__ y,
                                                      double *__restrict__ out)
{
    extern __shared__ double smem[];
    __shared__ Tables t;              // rhs / jacobian expect the descriptor in shared memory (see integrate_kernel)
    if (threadIdx.x == 0) t = t_arg;
    __syncthreads();
    const int N = t.n_sp, NR = t.n_rx;
    const size_t wd = work_doubles(N, NR, Grp<G>::NW, t.n_fo);
    Work w = carve(smem + (size_t)group_in_block<G>() * wd, N, NR, Grp<G>::NW, t.n_fo);
    const int lane = Grp<G>::lane();
    const int gpb = block_of<G>() / G;
    for (int s = blockIdx.x * gpb + group_in_block<G>(); s < n_states; s += gridDim.x * gpb) {
        for (int i = lane; i < N; i += G) w.y[i] = y[(size_t)s * N + i];
        Grp<G>::sync();
        if (JAC) {
            jacobian<G>(t, w.cs, P, w.y, w.Jm);
            for (int i = lane; i < N * N; i += G) out[(size_t)s * N * N + i] = w.Jm[i];
        } else {
            rhs<G>(t, w.cs, P, w.y, w.f0);
            for (int i = lane; i < N; i += G) out[(size_t)s * N + i] = w.f0[i];
        }
        Grp<G>::sync();
    }
}

// Batched LU solve hook: one warp per system, matrices staged column-major in shared memory.
__global__ void __launch_bounds__(32) lu_solve_kernel(int n, int batch, int is_complex, const double *__restrict__ A,
                                                      const double *__restrict__ b, double *__restrict__ x, int *info)
{
    extern __shared__ double smem[];
    double *Ar = smem, *Ai = Ar + (size_t)n * n, *br = Ai + (size_t)n * n, *bi = br + n;
    int *ip = reinterpret_cast<int *>(bi + n);
    const int lane = threadIdx.x;
    for (int s = blockIdx.x; s < batch; s += gridDim.x) {
        if (is_complex) {
            for (int e = lane; e < n * n; e += 32) {
                const int i = e / n, j = e % n;
                Ar[i + j * n] = A[((size_t)s * n * n + e) * 2];
                Ai[i + j * n] = A[((size_t)s * n * n + e) * 2 + 1];
            }
            for (int i = lane; i < n; i += 32) { br[i] = b[((size_t)s * n + i) * 2]; bi[i] = b[((size_t)s * n + i) * 2 + 1]; }
        } else {
            for (int e = lane; e < n * n; e += 32) {
                const int i = e / n, j = e % n;
                Ar[i + j * n] = A[(size_t)s * n * n + e];
            }
            for (int i = lane; i < n; i += 32) br[i] = b[(size_t)s * n + i];
        }
        __syncwarp();
        int ier;
        if (is_complex) {
            ier = lu_complex<32>(n, Ar, Ai, ip);
            __syncwarp();
            if (!ier) solve_complex_warp(n, Ar, Ai, ip, br, bi, lane);
        } else {
            ier = lu_real<32>(n, Ar, ip);
            __syncwarp();
            if (!ier) solve_real_warp(n, Ar, ip, br, lane);
        }
        __syncwarp();
        if (is_complex)
            for (int i = lane; i < n; i += 32) { x[((size_t)s * n + i) * 2] = br[i]; x[((size_t)s * n + i) * 2 + 1] = bi[i]; }
        else
            for (int i = lane; i < n; i += 32) x[(size_t)s * n + i] = br[i];
        if (info && lane == 0) info[s] = ier;
        __syncwarp();
    }
}

// The same hook for 16 < n <= 64 through the group kernels' routines (lu2_pair + solve2_pair, chem_device.cuh): one CTA
// of 128 threads per system.  The routines factor a real and a complex matrix side by side: a real system is given as
// both (zero imaginary parts), a complex one is paired with the identity.
__global__ void __launch_bounds__(128) lu2_solve_kernel(int n, int batch, int is_complex, const double *__restrict__ A,
                                                        const double *__restrict__ b, double *__restrict__ x, int *info)
{
    extern __shared__ double smem[];
    const int LD = n + 1;
    double *E1 = smem, *E2r = E1 + (size_t)n * LD, *E2i = E2r + (size_t)n * LD, *z1 = E2i + (size_t)n * LD, *z2 = z1 + n, *z3 = z2 + n;
    Lu2Aux x1, x2;
    x1.rdr = z3 + n; x1.rdi = nullptr; x2.rdr = x1.rdr + n; x2.rdi = x2.rdr + n;
    x1.perm = reinterpret_cast<int *>(x2.rdi + n); x1.rowk = x1.perm + n; x2.perm = x1.rowk + n; x2.rowk = x2.perm + n;
    const int tid = threadIdx.x;
    for (int s = blockIdx.x; s < batch; s += gridDim.x) {
        for (int e = tid; e < n * LD; e += 128) { E1[e] = 0.0; E2r[e] = 0.0; E2i[e] = 0.0; }
        __syncthreads();
        for (int e = tid; e < n * n; e += 128) {
            const int i = e / n, j = e % n;
            const size_t g = (size_t)s * n * n + e;
            if (is_complex) { E1[i + j * LD] = (i == j) ? 1.0 : 0.0; E2r[i + j * LD] = A[2 * g]; E2i[i + j * LD] = A[2 * g + 1]; }
            else { E1[i + j * LD] = A[g]; E2r[i + j * LD] = A[g]; }
        }
        for (int i = tid; i < n; i += 128) {
            const size_t g = (size_t)s * n + i;
            z1[i] = is_complex ? 0.0 : b[g];
            z2[i] = is_complex ? b[2 * g] : b[g];
            z3[i] = is_complex ? b[2 * g + 1] : 0.0;
        }
        __syncthreads();
        const int ier = (s & 1) ? lu2_pair<128>(n, LD, E1, x1, E2r, E2i, x2) : lu2_split(n, LD, E1, x1, E2r, E2i, x2);   // both forms are tested
        __syncthreads();
        if (!ier) {
            solve2_pair<128>(n, LD, E1, x1, z1, E2r, E2i, x2, z2, z3);
            for (int i = tid; i < n; i += 128) {
                const size_t g = (size_t)s * n + i;
                if (is_complex) { x[2 * g] = z2[i]; x[2 * g + 1] = z3[i]; } else x[g] = z1[i];
            }
        }
        if (info && tid == 0) info[s] = ier;
        __syncthreads();
    }
}

// The same hook for n <= 16 through the warp path's own routines (gj_warp_pair / solve_warp_pair, chem_warp.cuh):
// one warp per system, both half-warps are given the system (a real one with zero imaginary parts).
__global__ void __launch_bounds__(32) lu_solve_warp_kernel(int n, int batch, int is_complex, const double *__restrict__ A,
                                                           const double *__restrict__ b, double *__restrict__ x, int *info)
{
    extern __shared__ double smem[];
    const int LD = n | 1;
    double2 *Z = reinterpret_cast<double2 *>(smem), *bp = Z + 2 * n * LD;
    const int lane = threadIdx.x, h = lane >> 4, r = lane & 15;
    for (int s = blockIdx.x; s < batch; s += gridDim.x) {
        for (int e = lane; e < n * n; e += 32) {
            const size_t g = (size_t)s * n * n + e;
            const double2 v = is_complex ? make_double2(A[2 * g], A[2 * g + 1]) : make_double2(A[g], 0.0);
            Z[(e / n) * LD + e % n] = v;
            Z[n * LD + (e / n) * LD + e % n] = v;
        }
        __syncwarp();
        int myk = -1, src = lane;
        double rdr = 0.0, rdi = 0.0;
        const int ier = gj_warp_pair(Z, LD, n, myk, src, rdr, rdi);
        __syncwarp();
        if (info && lane == 0) info[s] = ier;
        if (!ier) {
            const size_t g = (size_t)s * n + (r < n ? r : 0);
            const double br = is_complex ? b[2 * g] : b[g], bi = is_complex ? b[2 * g + 1] : 0.0;
            const double2 v = solve_warp_pair(Z, LD, n, bp, myk, src, rdr, rdi, br, bi);
            if (h == 0 && r < n) {
                if (is_complex) { x[2 * g] = v.x; x[2 * g + 1] = v.y; } else x[g] = v.x;
            }
        }
        __syncwarp();
    }
}

}  // namespace

#include "chem_launch.inl"

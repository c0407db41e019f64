// chem_warp.cuh -- compact warp-per-state path for small mechanisms (N_sp <= 16, N_rx <= 32).
//
// One warp owns one state; control flow is uniform across the warp (divergence is the
// paper's first limiter).  Lane i (< N) holds component i of every stage / work vector in registers and
// owns ROW i of the matrices E1 = gamma/h I - J and E2 = (alpha + i beta)/h I - J, which live in shared
// memory (their storage is the paper's second limiter); rows are never moved, the pivot order
// is a permutation.  Lane i (< N_rx) owns reaction i: all transcendental work of a source-term evaluation
// is compiled by the mechanism compiler into "exp jobs"
//     exp(c0 + c1 ln T + c2/T + c3 T + c4 T^2 + c5 T^3 + c6 T^4)
// (forward rate, reverse rate with the equilibrium constant folded in, k0/kinf, the three Troe terms), two
// jobs per lane.  The code is deliberately compact (rolled loops, one out-of-line copy of every routine):
// the first version of this kernel was bound by instruction-cache misses (profiles/r1_generic_ncu.md).
#pragma once
#include "chem_radau.cuh"

namespace chem {

constexpr int kJobW = 8;     // doubles per job row (7 used)
constexpr int kJobs = 64;    // 2 rounds x 32 lanes
// fixed part of the staged table blob (doubles)
constexpr int kOffJobLo = 8, kOffJobHi = kOffJobLo + kJobs * kJobW, kOffSpLo = kOffJobHi + kJobs * kJobW;
constexpr int kOffSpHi = kOffSpLo + 16 * kJobW, kOffDesc = kOffSpHi + 16 * kJobW;   // desc: 32 lanes x 8 ints = 128 doubles
constexpr int kOffLists = kOffDesc + 128;

// Tables of the fast path: one blob in global memory, staged into shared memory once per CTA.
// blob[0..7] is a header of ints: {n_sp, n_rx, off_inc_nu, off_inc_rx, off_eff_dv, off_eff_sp, LD, 0} (offsets in doubles).
struct FastTables {
    int enabled;
    int n_sp, n_rx;
    int blob_doubles;
    double tmid;             // common NASA switch temperature
    const double *blob;
};

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ void warp_sum2(double &a, double &b)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, o);
        b += __shfl_xor_sync(0xffffffffu, b, o);
    }
}
__device__ __noinline__ double pow_ni(double a, double b) { return pow(a, b); }

// per-warp scratch layout (doubles): C[16] E[64] q[32] ys[16] then matrices
constexpr int kWsC = 0, kWsE = 16, kWsQ = 16 + kJobs, kWsYs = kWsQ + 32, kWsMat = kWsYs + 16;

// Source term for the state whose component `lane` is yc (lane 0: T, lanes 1..N-1: Y_1..Y_{N-1}).
// Returns component `lane` of f.  DESIGN.md R1-R5; same mathematics as rhs<G>() in chem_device.cuh.
// tab = staged table blob (shared), ws = this warp's scratch (shared).
__device__ __noinline__ double warp_rhs(const double *tab, double *ws, double tmid, double P, double yc)
{
    const int lane = threadIdx.x & 31;
    const int *hdr = reinterpret_cast<const int *>(tab);
    const int N = hdr[0];
    const int4 d0 = reinterpret_cast<const int4 *>(tab + kOffDesc)[2 * lane];       // slots, nus, type, jobs
    const int4 d1 = reinterpret_cast<const int4 *>(tab + kOffDesc)[2 * lane + 1];   // eff_lo, eff_hi, inc_lo, inc_hi
    double *C = ws + kWsC, *E = ws + kWsE, *q = ws + kWsQ;
    const double T = __shfl_sync(0xffffffffu, yc, 0);
    double Yk = __shfl_down_sync(0xffffffffu, yc, 1);     // species lane k holds Y_k = component k+1
    if (lane >= N - 1) Yk = 0.0;
    const bool lo = (T <= tmid);
    const double *spt = tab + (lo ? kOffSpLo : kOffSpHi);
    const double *spc = spt + (lane < N ? lane : 0) * kJobW;
    const double invWk = spc[7];
    double sY = Yk, sYW = Yk * invWk;
    warp_sum2(sY, sYW);
    const double YN = 1.0 - sY;                            // closure: last species
    if (lane == N - 1) Yk = YN;
    const double Wbar = 1.0 / (sYW + YN * spt[(N - 1) * kJobW + 7]);
    const double rho = P * Wbar / (kRerg * T);
    const double lnT = log(T), invT = 1.0 / T;
    const double Ck = rho * Yk * invWk;
    if (lane < N) C[lane] = Ck;
    // two exp jobs per lane
    const double *jt = tab + (lo ? kOffJobLo : kOffJobHi);
    double Ej[2];
#pragma unroll 1
    for (int r = 0; r < 2; r++) {
        const double *c = jt + (32 * r + lane) * kJobW;
        Ej[r] = exp(c[0] + c[1] * lnT + c[2] * invT + T * (c[3] + T * (c[4] + T * (c[5] + T * c[6]))));
        E[32 * r + lane] = Ej[r];
    }
    __syncwarp();
    // rate of progress of reaction `lane`
    double qi = 0.0;
    const int type = d0.z;
    if (type >= 0) {
        double Rf = E[lane], Rr = E[32 + lane];
#pragma unroll
        for (int sl = 0; sl < 6; sl++) {
            const int sp = (d0.x >> (5 * sl)) & 31, nu = (d0.y >> (2 * sl)) & 3;
            const double pw = powi(C[sp], nu);
            if (sl < 3) Rf *= pw; else Rr *= pw;
        }
        double c = 1.0;
        if (type != 0) {
            const double *eff_dv = tab + hdr[4];
            const int *eff_sp = reinterpret_cast<const int *>(tab + hdr[5]);
            double M = P / (kRerg * T);
            for (int p = d1.x; p < d1.y; p++) M += eff_dv[p] * C[eff_sp[p]];
            if (type == 1) {
                c = M;
            } else {
                const double Pr = E[d0.w & 255] * M;
                double F = 1.0;
                if (type == 3) {
                    const int ts = (d0.w >> 8) & 255;
                    const double Fc = E[ts] + E[ts + 1] + E[ts + 2];
                    const double L = log10(Fc);
                    const double At = log10(Pr) - 0.4 - 0.67 * L;
                    const double Bt = 0.75 - 1.27 * L - 0.14 * At;
                    const double x = At / Bt;
                    F = exp10(L / (1.0 + x * x));
                }
                c = Pr / (1.0 + Pr) * F;
            }
        }
        qi = c * (Rf - Rr);
    }
    q[lane] = qi;
    __syncwarp();
    // species production rates, temperature equation
    const double *inc_nu = tab + hdr[2];
    const int *inc_rx = reinterpret_cast<const int *>(tab + hdr[3]);
    double w = 0.0;
    for (int p = d1.z; p < d1.w; p++) w += inc_nu[p] * q[inc_rx[p]];
    const double cpR = spc[0] + T * (spc[1] + T * (spc[2] + T * (spc[3] + T * spc[4])));
    const double hRT = spc[0] + T * (spc[1] * 0.5 + T * (spc[2] * (1.0 / 3.0) + T * (spc[3] * 0.25 + T * (spc[4] * 0.2)))) + spc[5] * invT;
    double hw = (lane < N) ? hRT * w : 0.0, ccp = (lane < N) ? Ck * cpR : 0.0;
    warp_sum2(hw, ccp);
    const double Ydot = spc[6] * w / rho;                 // W_k wdot_k / rho in species lane k
    double f = __shfl_up_sync(0xffffffffu, Ydot, 1);      // component k+1
    if (lane == 0) f = -T * hw / ccp;
    __syncwarp();
    return f;
}

// ---------------------------------------------------------------------------- LU with rows owned by lanes
// exact argmax over lanes of a non-negative key v (inactive lanes pass -1): highest 32 bits first, low word
// only on ties; lowest lane wins exact ties.  Returns -1 if the maximum is not > 0.
__device__ __forceinline__ int warp_argmax(double v)
{
    const bool act = v >= 0.0;
    const unsigned hi = act ? (unsigned)__double2hiint(v) : 0u;
    const unsigned m = __reduce_max_sync(0xffffffffu, hi);
    unsigned cand = __ballot_sync(0xffffffffu, act && hi == m);
    if (__popc(cand) != 1) {
        const unsigned lo = (act && hi == m) ? (unsigned)__double2loint(v) : 0u;
        const unsigned m2 = __reduce_max_sync(0xffffffffu, lo);
        cand = __ballot_sync(0xffffffffu, act && hi == m && lo == m2);
        if (m == 0u && m2 == 0u) return -1;
    }
    if (cand == 0u) return -1;
    return __ffs(cand) - 1;
}

// Real LU, A[i*LD + j] in shared memory, row i owned by lane i.  perm[k] = pivot lane of step k; myk = the
// step at which this lane's row was the pivot row; rdiag = 1/U_kk held by the pivot lane of step k.
__device__ __noinline__ int lu_warp_real(double *A, int LD, int N, int *perm, int &myk_out, double &rdiag_out)
{
    const int lane = threadIdx.x & 31;
    double *row = A + (lane < N ? lane : 0) * LD;
    int myk = -1;
    double rdiag = 0.0;
    for (int k = 0; k < N; k++) {
        const bool act = (lane < N) && (myk < 0);
        const double ak = row[k];
        const int p = warp_argmax(act ? fabs(ak) : -1.0);
        if (p < 0) return k + 1;
        const double *prow = A + p * LD;
        const double pvv = prow[k];
        if (!isfinite(pvv)) return k + 1;
        const double rp = 1.0 / pvv;
        if (lane == 0) perm[k] = p;
        if (lane == p) { myk = k; rdiag = rp; }
        if (act && lane != p) {
            const double l = ak * rp;
            row[k] = l;
            for (int j = k + 1; j < N; j++) row[j] = fma(-l, prow[j], row[j]);
        }
        __syncwarp();
    }
    myk_out = myk;
    rdiag_out = rdiag;
    return 0;
}

__device__ __noinline__ int lu_warp_complex(double *Ar, double *Ai, int LD, int N, int *perm, int &myk_out, double &rdr_out,
                                            double &rdi_out)
{
    const int lane = threadIdx.x & 31;
    const int off = (lane < N ? lane : 0) * LD;
    double *rr = Ar + off, *ri = Ai + off;
    int myk = -1;
    double rdr = 0.0, rdi = 0.0;
    for (int k = 0; k < N; k++) {
        const bool act = (lane < N) && (myk < 0);
        const double akr = rr[k], aki = ri[k];
        const int p = warp_argmax(act ? fabs(akr) + fabs(aki) : -1.0);
        if (p < 0) return k + 1;
        const double *pr_ = Ar + p * LD, *pi_ = Ai + p * LD;
        const double pr = pr_[k], pi = pi_[k];
        const double den = 1.0 / (pr * pr + pi * pi);
        if (!isfinite(den)) return k + 1;
        const double qr = pr * den, qi = -pi * den;       // 1 / pivot
        if (lane == 0) perm[k] = p;
        if (lane == p) { myk = k; rdr = qr; rdi = qi; }
        if (act && lane != p) {
            const double lr = akr * qr - aki * qi, li = akr * qi + aki * qr;
            rr[k] = lr;
            ri[k] = li;
            for (int j = k + 1; j < N; j++) {
                const double ur = pr_[j], ui = pi_[j];
                rr[j] = fma(-lr, ur, fma(li, ui, rr[j]));
                ri[j] = fma(-lr, ui, fma(-li, ur, ri[j]));
            }
        }
        __syncwarp();
    }
    myk_out = myk;
    rdr_out = rdr;
    rdi_out = rdi;
    return 0;
}

// Solves: b = component `lane` of the right-hand side (original row order); returns component `lane` of x.
__device__ __noinline__ double solve_warp_real(const double *A, int LD, int N, const int *perm, int myk, double rdiag, double b)
{
    const int lane = threadIdx.x & 31;
    const double *row = A + (lane < N ? lane : 0) * LD;
    for (int k = 0; k < N - 1; k++) {
        const double bk = __shfl_sync(0xffffffffu, b, perm[k]);
        if (myk > k) b = fma(-row[k], bk, b);
    }
    double x = 0.0;
    for (int k = N - 1; k >= 0; k--) {
        const double xk = __shfl_sync(0xffffffffu, b * rdiag, perm[k]);
        if (myk >= 0 && myk < k) b = fma(-row[k], xk, b);
        if (lane == k) x = xk;
    }
    return x;
}

__device__ __noinline__ double2 solve_warp_complex(const double *Ar, const double *Ai, int LD, int N, const int *perm, int myk,
                                                   double rdr, double rdi, double br, double bi)
{
    const int lane = threadIdx.x & 31;
    const int off = (lane < N ? lane : 0) * LD;
    const double *rr = Ar + off, *ri = Ai + off;
    for (int k = 0; k < N - 1; k++) {
        const int p = perm[k];
        const double xr = __shfl_sync(0xffffffffu, br, p), xi = __shfl_sync(0xffffffffu, bi, p);
        if (myk > k) {
            const double lr = rr[k], li = ri[k];
            br = fma(-lr, xr, fma(li, xi, br));
            bi = fma(-lr, xi, fma(-li, xr, bi));
        }
    }
    double sr = 0.0, si = 0.0;
    for (int k = N - 1; k >= 0; k--) {
        const int p = perm[k];
        const double vr = br * rdr - bi * rdi, vi = br * rdi + bi * rdr;
        const double xr = __shfl_sync(0xffffffffu, vr, p), xi = __shfl_sync(0xffffffffu, vi, p);
        if (myk >= 0 && myk < k) {
            const double ur = rr[k], ui = ri[k];
            br = fma(-ur, xr, fma(ui, xi, br));
            bi = fma(-ur, xi, fma(-ui, xr, bi));
        }
        if (lane == k) { sr = xr; si = xi; }
    }
    return make_double2(sr, si);
}

}  // namespace chem

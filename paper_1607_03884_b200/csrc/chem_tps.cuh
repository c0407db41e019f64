// chem_tps.cuh -- thread-per-state path for small mechanisms (N_sp <= 16, N_rx <= 32): device routines.
//
// The paper's own GPU mapping is one CUDA thread per IVP, and it names the two things that
// limit it: thread divergence (L184, L194) and the storage of the Jacobian and its factors (L182).  This is that
// mapping rebuilt for sm_100a:
//   * every lane of a warp owns one state and runs the Radau IIA controller as a STATE MACHINE; a warp executes the
//     phases (Newton iteration, error estimate, source term, Jacobian, factorisation) one after the other, each for the
//     lanes that want it, and a lane that finishes its state pulls the next one from the work queue at once -- so the
//     spread of step counts between states (Eq. 3) costs nothing, and what is left of divergence is the share of lanes
//     that sit out a phase;
//   * all data of a lane is addressed [element][lane] (structure of arrays across the warp): every access of a warp is
//     one coalesced 256-byte row, in shared memory (work vectors, conflict-free) and in global memory (the matrices,
//     L2-resident); element indices are uniform across the warp except for the row interchanges of partial pivoting;
//   * the device routines below have no cross-lane communication at all (no shuffles, no reductions, no barriers), so any
//     subset of the lanes may call them; the kernel (chem_tps.cu) puts a __syncwarp() in front of every phase -- without it
//     the compiler lets the lanes that skip a phase run ahead into the next one and every phase runs twice, with
//     complementary halves of the warp -- and one CTA barrier per pass, so that the warps of a CTA are in the same phase at
//     the same time and share their instruction-cache fills.
// The arithmetic is that of chem_warp.cuh (exp-job tables of the mechanism compiler, R1-R12) with plain LU +
// triangular solves, left-looking so that each factor entry is written once.
#pragma once
#include "chem_common.cuh"

namespace chem {
namespace tps {

typedef unsigned long long u64;

// lane-private element e of an array whose rows are 32 lanes wide
#define TL(p, e) (p)[(e) * 32]

// L2 eviction priorities for the lane-private global workspace ("storage of the Jacobian matrix and/or
// factorized forms ... cause many slow global memory accesses").  The LU factors of all resident lanes (4 KB each, 154 MB
// at N = 13) are re-read by every triangular solve and do not fit the 126 MB L2 together: read round-robin they evict
// each other and most solves stream from HBM.  So the factors of `keep` warps out of every 8 are tagged evict_last -- that
// subset fits and stays resident -- and the factors of the other warps, like J, are tagged evict_first: they stream
// through without displacing the resident set (profiles/r3_tps_config1.md).
__device__ __forceinline__ u64 l2_policy(bool keep)
{
    u64 last, first;
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(last));
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(first));
    return keep ? last : first;
}
__device__ __forceinline__ double ldp(const double *p, u64 pol)
{
    double v;
    asm volatile("ld.global.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(p), "l"(pol) : "memory");
    return v;
}
__device__ __forceinline__ double2 ldp(const double2 *p, u64 pol)
{
    double2 v;
    asm volatile("ld.global.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol) : "memory");
    return v;
}
__device__ __forceinline__ void stp(double *p, double v, u64 pol)
{
    asm volatile("st.global.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(p), "d"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ void stp(double2 *p, double2 v, u64 pol)
{
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}
// the same access pattern as TL with a cache policy
#define TLP(p, e, pol) ldp(&(p)[(e) * 32], pol)

// Shared-memory elements per lane: y[N], z1..z3[3N], C[N+1], U[max(N_rx, 2N+1)] (q of the source term; row and S of the
// Jacobian); z doubles as the column scratch of the factorisation.  Global elements per lane (L2-resident workspace):
// J[N^2], E1[N^2], E2[N^2] complex, f0[N], cont[3N], w1..w3[3N], a1..a3[3N], the Jacobian's reaction records[4 N_rx].
struct Lay {
    int N, NR, n_sm, n_gw;
};
__host__ __device__ inline int oZ(int N) { return N; }
__host__ __device__ inline int oC(int N) { return 4 * N; }
__host__ __device__ inline int oU(int N) { return 5 * N + 1; }
__host__ __device__ inline int gE1(int N) { return N * N; }
__host__ __device__ inline int gE2(int N) { return 2 * N * N; }   // in doubles; E2 is addressed as double2 from here
__host__ __device__ inline int gF0(int N) { return 4 * N * N; }
__host__ __device__ inline int gCT(int N) { return 4 * N * N + N; }
__host__ __device__ inline int gW(int N) { return 4 * N * N + 4 * N; }
__host__ __device__ inline int gA(int N) { return 4 * N * N + 7 * N; }
__host__ __device__ inline int gR(int N) { return 4 * N * N + 10 * N; }
__host__ __device__ inline Lay make_lay(int N, int NR)
{
    Lay L;
    L.N = N; L.NR = NR;
    L.n_sm = oU(N) + (NR > 2 * N + 1 ? NR : 2 * N + 1);
    L.n_gw = gR(N) + 4 * NR;
    return L;
}

__device__ __forceinline__ double nan_d() { return __longlong_as_double(0x7ff8000000000000LL); }

// exp(x) as exp_f (chem_math.cuh: same range reduction, same degree-13 Taylor polynomial, same tails) with the
// polynomial evaluated by Estrin's scheme: a lane has only its own instruction stream to hide the 8-cycle DFMA latency
// with, and Horner's rule is a chain of 13 dependent DFMAs; this is 5 levels deep for 4 more multiplications.
__device__ __forceinline__ double exp_e(double x)
{
    const double t = fma(x, 1.4426950408889634074, 6755399441055744.0);
    const int n = __double2loint(t);
    const double fn = t - 6755399441055744.0;
    double r = fma(fn, -6.93147180369123816490e-01, x);
    r = fma(fn, -1.90821492927058770002e-10, r);
    const double r2 = r * r, r4 = r2 * r2, r8 = r4 * r4;
    const double p01 = fma(kExpC[1], r, kExpC[0]), p23 = fma(kExpC[3], r, kExpC[2]), p45 = fma(kExpC[5], r, kExpC[4]);
    const double p67 = fma(kExpC[7], r, kExpC[6]), p89 = fma(kExpC[9], r, kExpC[8]), pab = fma(kExpC[11], r, kExpC[10]);
    const double pcd = fma(kExpC[13], r, kExpC[12]);
    const double q0 = fma(p23, r2, p01), q1 = fma(p67, r2, p45), q2 = fma(pab, r2, p89);
    const double s0 = fma(q1, r4, q0), s1 = fma(pcd, r4, q2);
    double p = fma(s1, r8, s0);
    const int n1 = n >> 1, n2 = n - n1;
    p *= __hiloint2double((1023 + n1) << 20, 0);
    p *= __hiloint2double((1023 + n2) << 20, 0);
    if (x < -700.0) p = 0.0;
    if (x > 709.0) p = __longlong_as_double(0x7ff0000000000000LL);
    return p;
}

// ------------------------------------------------------------------------------------------------ source term
// f(T, Y; P) at the state y + vs * v (R1-R5; same mathematics as warp_rhs_body, chem_warp.cuh), all lane-private:
// y = sm[0..N), v and the result `out` anywhere (shared or global; v is consumed before the scratch is written).
// tab = staged table blob (shared, read with uniform indices).
static __device__ __noinline__ void rhs(const double *tab, double *sm, int N, int NR, double tmid, double P, double invP,
                                 const double *v, double vs, double *out)
{
    const int *hdr = reinterpret_cast<const int *>(tab);
    const int4 *desc = reinterpret_cast<const int4 *>(tab + kOffDesc);
    const double *y = sm;
    double *C = sm + oC(N) * 32, *q = sm + oU(N) * 32;
    const double *spw = tab + kOffSpLo;                       // W and 1/W are the same in both NASA ranges
    const double T = fma(vs, TL(v, 0), TL(y, 0));
    double sY = 0.0, sYW = 0.0;
#pragma unroll 4
    for (int k = 0; k < N - 1; k++) {
        const double Yk = fma(vs, TL(v, k + 1), TL(y, k + 1));
        sY += Yk;
        sYW = fma(Yk, spw[k * kJobW + 7], sYW);
        TL(C, k) = Yk;
    }
    const double YN = 1.0 - sY;                               // closure: last species
    TL(C, N - 1) = YN;
    const double sW = fma(YN, spw[(N - 1) * kJobW + 7], sYW); // 1 / Wbar
    const double Wbar = rcp_f(sW), invT = rcp_f(T);
    const double rho = P * Wbar * invT * (1.0 / kRerg), inv_rho = kRerg * T * sW * invP;
    const double lnT = T > 0.0 ? log_f(T) : nan_d();          // a Newton iterate may overshoot to T <= 0: failed step (R11)
#pragma unroll 4
    for (int k = 0; k < N; k++) TL(C, k) = rho * TL(C, k) * spw[k * kJobW + 7];
    TL(C, N) = 1.0;                                           // unity factor of unused slots
    const bool lo = T <= tmid;
    const double *jt = tab + (lo ? kOffJobLo : kOffJobHi);
    // mass-action part of every reaction: two exp jobs (k_f, k_r with K_c folded in) and three factors per side; two
    // reactions per trip, all table and concentration reads before the stores, so that four exponentials overlap
    {
        auto ropa = [&](int i, double &kf_arg, double &kr_arg, double &pf, double &pr) {
            kf_arg = job_arg(jt + i * kJobW, T, lnT, invT);
            kr_arg = job_arg(jt + (32 + i) * kJobW, T, lnT, invT);
            const int sl = desc[i].x;
            pf = TL(C, min(sl & 31, N)) * TL(C, min((sl >> 5) & 31, N)) * TL(C, min((sl >> 10) & 31, N));
            pr = TL(C, min((sl >> 15) & 31, N)) * TL(C, min((sl >> 20) & 31, N)) * TL(C, min((sl >> 25) & 31, N));
        };
        int i = 0;
#pragma unroll 1
        for (; i + 1 < NR; i += 2) {
            double a0, b0, f0, r0, a1, b1, f1, r1;
            ropa(i, a0, b0, f0, r0);
            ropa(i + 1, a1, b1, f1, r1);
            const double q0 = exp_e(a0) * f0 - exp_e(b0) * r0, q1 = exp_e(a1) * f1 - exp_e(b1) * r1;
            TL(q, i) = q0;
            TL(q, i + 1) = q1;
        }
        if (i < NR) {
            double a0, b0, f0, r0;
            ropa(i, a0, b0, f0, r0);
            TL(q, i) = exp_e(a0) * f0 - exp_e(b0) * r0;
        }
    }
    // third-body and falloff factors (the reaction type is uniform across the warp)
    const double Ctot = P * invT * (1.0 / kRerg);
    const double *eff_dv = tab + hdr[4];
    const int *eff_sp = reinterpret_cast<const int *>(tab + hdr[5]);
#pragma unroll 1
    for (int i = 0; i < NR; i++) {
        const int4 d0 = desc[i];
        if (d0.z <= 0) continue;
        const int4 d1 = desc[32 + i];
        double cm = Ctot;
#pragma unroll 1
        for (int p = d1.x; p < d1.y; p++) cm = fma(eff_dv[p], TL(C, eff_sp[p]), cm);
        if (d0.z >= 2) {
            const double Pr = exp_e(job_arg(jt + (d0.w & 255) * kJobW, T, lnT, invT)) * cm;
            double F = 1.0;
            if (d0.z == 3) {
                const double *c = jt + ((d0.w >> 8) & 255) * kJobW;
                const double Fc = exp_e(job_arg(c, T, lnT, invT)) + exp_e(job_arg(c + kJobW, T, lnT, invT)) +
                                  exp_e(job_arg(c + 2 * kJobW, T, lnT, invT));
                const double lg = log_f(Fc) * kInvLn10, lPr = log_f(Pr) * kInvLn10;
                const double At = lPr - 0.4 - 0.67 * lg;
                const double x = At * rcp_f(0.75 - 1.27 * lg - 0.14 * At);
                F = exp_e(kLn10 * lg * rcp_f(fma(x, x, 1.0)));
            }
            cm = Pr * rcp_f(1.0 + Pr) * F;
        }
        TL(q, i) *= cm;
    }
    // species production rates, temperature equation
    const int2 *inc = reinterpret_cast<const int2 *>(tab + hdr[3]);
    const double *spt = tab + (lo ? kOffSpLo : kOffSpHi);
    double hw = 0.0, ccp = 0.0;
#pragma unroll 1
    for (int k = 0; k < N; k++) {
        const int4 d1 = desc[32 + k];
        double w0 = 0.0, w1 = 0.0;
        int p = d1.z;
#pragma unroll 2
        for (; p + 1 < d1.w; p += 2) {
            const int2 e0 = inc[p], e1 = inc[p + 1];
            w0 = fma((double)e0.y, TL(q, e0.x), w0);
            w1 = fma((double)e1.y, TL(q, e1.x), w1);
        }
        if (p < d1.w) { const int2 e0 = inc[p]; w0 = fma((double)e0.y, TL(q, e0.x), w0); }
        const double w = w0 + w1;
        const double *sc = spt + k * kJobW;
        const double cpR = sc[0] + T * (sc[1] + T * (sc[2] + T * (sc[3] + T * sc[4])));
        const double hRT = sc[0] + T * (sc[1] * 0.5 + T * (sc[2] * (1.0 / 3.0) + T * (sc[3] * 0.25 + T * (sc[4] * 0.2)))) + sc[5] * invT;
        hw = fma(hRT, w, hw);
        ccp = fma(TL(C, k), cpR, ccp);
        if (k < N - 1) TL(out, k + 1) = sc[6] * w * inv_rho;
    }
    TL(out, 0) = -T * hw * rcp_f(ccp);
}

// ------------------------------------------------------------------------------------------------ analytical Jacobian
// J[i*N + j] = d f_i / d y_j at y -> global gJ (R6; the formulation of warp_jacobian, chem_warp.cuh).  Pass 1
// leaves four numbers per reaction (c k_f, -c k_r, dq/dT at constant C, dq/d[M]) in the lane's global workspace; pass 2 builds d wdot_k / d C row by row in a lane-private row buffer, applies the chain rule
// C -> (T, Y) and writes row k + 1 of J straight to global memory: N^2 global stores, no global read-modify-write.
static __device__ __noinline__ void jacobian(const double *tab, double *sm, double *gJ, double *rd, int N, int NR, double tmid, double P,
                                      double invP)
{
    const int *hdr = reinterpret_cast<const int *>(tab);
    const int4 *desc = reinterpret_cast<const int4 *>(tab + kOffDesc);
    const double *y = sm;
    double *C = sm + oC(N) * 32, *row = sm + oU(N) * 32, *S = row + (N + 1) * 32;   // rd: [4][NR] in global memory
    const double *spw = tab + kOffSpLo;
    const double *eff_dv = tab + hdr[4];
    const int *eff_sp = reinterpret_cast<const int *>(tab + hdr[5]);
    const int2 *inc = reinterpret_cast<const int2 *>(tab + hdr[3]);
    const double T = TL(y, 0);
    double sY = 0.0, sYW = 0.0;
#pragma unroll 4
    for (int k = 0; k < N - 1; k++) {
        const double Yk = TL(y, k + 1);
        sY += Yk;
        sYW = fma(Yk, spw[k * kJobW + 7], sYW);
        TL(C, k) = Yk;
    }
    const double YN = 1.0 - sY;
    TL(C, N - 1) = YN;
    const double invWN = spw[(N - 1) * kJobW + 7];
    const double sW = fma(YN, invWN, sYW);
    const double Wbar = rcp_f(sW), invT = rcp_f(T);
    const double rho = P * Wbar * invT * (1.0 / kRerg), inv_rho = kRerg * T * sW * invP;
    const double lnT = T > 0.0 ? log_f(T) : nan_d();
#pragma unroll 4
    for (int k = 0; k < N; k++) TL(C, k) = rho * TL(C, k) * spw[k * kJobW + 7];
    TL(C, N) = 1.0;
    const bool lo = T <= tmid;
    const double *jt = tab + (lo ? kOffJobLo : kOffJobHi);
    const double Ctot = P * invT * (1.0 / kRerg);
    // pass 1: per-reaction records
#pragma unroll 1
    for (int i = 0; i < NR; i++) {
        const int4 d0 = desc[i];
        const int sl = d0.x;
        const double kf = exp_e(job_arg(jt + i * kJobW, T, lnT, invT));
        const double kr = exp_e(job_arg(jt + (32 + i) * kJobW, T, lnT, invT));
        const double dlnkf = job_darg(jt + i * kJobW, T, invT), dlnkr = job_darg(jt + (32 + i) * kJobW, T, invT);
        const double Rf = kf * (TL(C, min(sl & 31, N)) * TL(C, min((sl >> 5) & 31, N)) * TL(C, min((sl >> 10) & 31, N)));
        const double Rr = kr * (TL(C, min((sl >> 15) & 31, N)) * TL(C, min((sl >> 20) & 31, N)) * TL(C, min((sl >> 25) & 31, N)));
        const double rnet = Rf - Rr;
        double c = 1.0, dc_dT = 0.0, dc_dM = 0.0;
        if (d0.z > 0) {
            const int4 d1 = desc[32 + i];
            double M = Ctot;
#pragma unroll 1
            for (int p = d1.x; p < d1.y; p++) M = fma(eff_dv[p], TL(C, eff_sp[p]), M);
            c = M;
            dc_dM = 1.0;
            if (d0.z >= 2) {
                const int ks = d0.w & 255;
                const double k0k = exp_e(job_arg(jt + ks * kJobW, T, lnT, invT)), Pr = k0k * M;
                const double dlnPr = job_darg(jt + ks * kJobW, T, invT);
                double F = 1.0, dF_dT = 0.0, dF_dPr = 0.0;
                if (d0.z == 3) {
                    const double *cj = jt + ((d0.w >> 8) & 255) * kJobW;
                    const double e3 = exp_e(job_arg(cj, T, lnT, invT)), e1 = exp_e(job_arg(cj + kJobW, T, lnT, invT));
                    const double e2 = exp_e(job_arg(cj + 2 * kJobW, T, lnT, invT));
                    const double Fc = e3 + e1 + e2;
                    const double dFc = e3 * job_darg(cj, T, invT) + e1 * job_darg(cj + kJobW, T, invT) + e2 * job_darg(cj + 2 * kJobW, T, invT);
                    const double L = log_f(Fc) * kInvLn10, dL = dFc * rcp_f(Fc) * kInvLn10;
                    const double At = log_f(Pr) * kInvLn10 - 0.4 - 0.67 * L;
                    const double Bt = 0.75 - 1.27 * L - 0.14 * At, rB = rcp_f(Bt);
                    const double x = At * rB, rden = rcp_f(fma(x, x, 1.0));
                    F = exp_e(kLn10 * L * rden);
                    const double dA_T = dlnPr * kInvLn10 - 0.67 * dL, dB_T = -1.27 * dL - 0.14 * dA_T;
                    const double dx_T = (dA_T * Bt - At * dB_T) * rB * rB;
                    const double dx_P = rcp_f(Pr) * kInvLn10 * (Bt + 0.14 * At) * rB * rB;
                    const double wF = -L * 2.0 * x * rden * rden;
                    dF_dT = F * kLn10 * (dL * rden + wF * dx_T);
                    dF_dPr = F * kLn10 * wF * dx_P;
                }
                const double op = rcp_f(1.0 + Pr);
                c = Pr * op * F;
                dc_dT = Pr * dlnPr * op * op * F + Pr * op * dF_dT;
                dc_dM = (op * op * F + Pr * op * dF_dPr) * k0k;
            }
        }
        TL(rd, i) = c * kf;
        TL(rd, NR + i) = -c * kr;
        TL(rd, 2 * NR + i) = dc_dT * rnet + c * (Rf * dlnkf - Rr * dlnkr);
        TL(rd, 3 * NR + i) = d0.z > 0 ? dc_dM * rnet : 0.0;
    }
    // pass 2: rows
    const double *spt = tab + (lo ? kOffSpLo : kOffSpHi);
#pragma unroll 4
    for (int j = 0; j < N; j++) TL(S, j) = 0.0;
    double hw = 0.0, ccp = 0.0, cpw = 0.0, cdcp = 0.0;
#pragma unroll 1
    for (int k = 0; k < N; k++) {
#pragma unroll 4
        for (int l = 0; l <= N; l++) TL(row, l) = 0.0;
        const int4 dk = desc[32 + k];
        double wd = 0.0, dwT = 0.0, u = 0.0;
#pragma unroll 1
        for (int p = dk.z; p < dk.w; p++) {
            const int2 e = inc[p];
            const int i = e.x;
            const double nu = (double)e.y;
            const int4 e0 = desc[i];
            const int sl = e0.x;
            const int f0 = min(sl & 31, N), f1 = min((sl >> 5) & 31, N), f2 = min((sl >> 10) & 31, N);
            const int f3 = min((sl >> 15) & 31, N), f4 = min((sl >> 20) & 31, N), f5 = min((sl >> 25) & 31, N);
            const double c0 = TL(C, f0), c1 = TL(C, f1), c2 = TL(C, f2), c3 = TL(C, f3), c4 = TL(C, f4), c5 = TL(C, f5);
            const double ckf = nu * TL(rd, i), ckr = nu * TL(rd, NR + i);
            const double a12 = ckf * c1 * c2, b45 = ckr * c4 * c5;
            wd += a12 * c0 + b45 * c3;                         // nu q_i
            dwT = fma(nu, TL(rd, 2 * NR + i), dwT);
            TL(row, f0) += a12;
            TL(row, f1) += ckf * c0 * c2;
            TL(row, f2) += ckf * c0 * c1;
            TL(row, f3) += b45;
            TL(row, f4) += ckr * c3 * c5;
            TL(row, f5) += ckr * c3 * c4;
            if (e0.z > 0) {
                const int4 e1 = desc[32 + i];
                const double vv = nu * TL(rd, 3 * NR + i);
                u += vv;
#pragma unroll 1
                for (int pe = e1.x; pe < e1.y; pe++) TL(row, eff_sp[pe]) = fma(vv, eff_dv[pe], TL(row, eff_sp[pe]));
            }
        }
        double GC = 0.0;
#pragma unroll 4
        for (int l = 0; l < N; l++) GC = fma(TL(row, l), TL(C, l), GC);
        const double GN = TL(row, N - 1) * invWN;
#pragma unroll 1
        for (int j = N - 1; j >= 1; j--) {
            const double iw = spw[(j - 1) * kJobW + 7];
            TL(row, j) = -Wbar * (iw - invWN) * GC + rho * (TL(row, j - 1) * iw - GN);
        }
        TL(row, 0) = dwT - (GC + u * Ctot) * invT;
        const double *sc = spt + k * kJobW;
        const double cpR = sc[0] + T * (sc[1] + T * (sc[2] + T * (sc[3] + T * sc[4])));
        const double dcpR = sc[1] + T * (2.0 * sc[2] + T * (3.0 * sc[3] + T * (4.0 * sc[4])));
        const double hRT = sc[0] + T * (sc[1] * 0.5 + T * (sc[2] * (1.0 / 3.0) + T * (sc[3] * 0.25 + T * (sc[4] * 0.2)))) + sc[5] * invT;
        const double Ck = TL(C, k);
        hw = fma(hRT, wd, hw); ccp = fma(Ck, cpR, ccp); cpw = fma(cpR, wd, cpw); cdcp = fma(Ck, dcpR, cdcp);
        const double Wr = sc[6] * inv_rho;
#pragma unroll 2
        for (int j = 0; j < N; j++) {
            const double r = TL(row, j);
            TL(S, j) = fma(hRT, r, TL(S, j));
            if (k < N - 1) {
                const double dlnrho = j == 0 ? -invT : -Wbar * (spw[(j - 1) * kJobW + 7] - invWN);
                TL(gJ, (k + 1) * N + j) = Wr * (r - wd * dlnrho);
            }
        }
    }
    const double rccp = rcp_f(ccp);
    const double Tdot = -T * hw * rccp;
    const double cpN = spt[(N - 1) * kJobW] + T * (spt[(N - 1) * kJobW + 1] + T * (spt[(N - 1) * kJobW + 2] +
                       T * (spt[(N - 1) * kJobW + 3] + T * spt[(N - 1) * kJobW + 4])));
#pragma unroll 1
    for (int j = 0; j < N; j++) {
        double dlnrho, drcp;
        if (j == 0) {
            dlnrho = -invT;
            drcp = -ccp * invT + cdcp;
        } else {
            const double *sc = spt + (j - 1) * kJobW;
            const double iw = spw[(j - 1) * kJobW + 7];
            const double cpj = sc[0] + T * (sc[1] + T * (sc[2] + T * (sc[3] + T * sc[4])));
            dlnrho = -Wbar * (iw - invWN);
            drcp = dlnrho * ccp + rho * (cpj * iw - cpN * invWN);
        }
        TL(gJ, j) = -(T * TL(S, j) + (j == 0 ? cpw : 0.0)) * rccp - Tdot * drcp * rccp;
    }
}

// ------------------------------------------------------------------------------------------------ LU and solves
// Both factorisations of a Radau step, left-looking, in one pass over the columns of J:
//   E1 = fac1 I - J (real) and E2 = (alphn + i betan) I - J (complex), column-major in global memory, unit lower factor
//   below the diagonal, U above it, the RECIPROCAL of the pivot on the diagonal; LAPACK row order (rows are swapped
//   physically, only by the lanes that pivot off the diagonal), pivot rows packed four bits per step in ip1 / ip2.
// Column j is loaded from J once, brought up to date in a lane-private shared-memory column (col: 3N entries) with the
// finished columns k < j -- the same operations in the same order as right-looking elimination, but every factor entry
// is written once -- then the pivot is searched (|re| + |im| for the complex matrix, first maximum wins: DESIGN.md R10).
// Returns 0, or j + 1 if a matrix has no usable pivot in column j or J is not finite.
static __device__ __noinline__ int lu_pair(const double *gJ, double *g1, double2 *g2, double *col, int N, double fac1, double alphn,
                                    double betan, u64 &ip1_out, u64 &ip2_out)
{
    double *c1 = col, *cr = col + N * 32, *ci = col + 2 * N * 32;
    u64 ip1 = 0, ip2 = 0;
    int ier = 0;
#pragma unroll 1
    for (int j = 0; j < N; j++) {
        bool bad = false;
#pragma unroll 4
        for (int i = 0; i < N; i++) {
            const double v = -TL(gJ, i * N + j);
            bad |= !isfinite(v);
            TL(c1, i) = v; TL(cr, i) = v; TL(ci, i) = 0.0;
        }
        TL(c1, j) += fac1; TL(cr, j) += alphn; TL(ci, j) = betan;
        // interchanges of the finished steps
#pragma unroll 1
        for (int k = 0; k < j; k++) {
            const int p1 = (int)(ip1 >> (4 * k)) & 15, p2 = (int)(ip2 >> (4 * k)) & 15;
            if (p1 != k) { const double t = TL(c1, k); TL(c1, k) = TL(c1, p1); TL(c1, p1) = t; }
            if (p2 != k) {
                const double t = TL(cr, k), s = TL(ci, k);
                TL(cr, k) = TL(cr, p2); TL(ci, k) = TL(ci, p2);
                TL(cr, p2) = t; TL(ci, p2) = s;
            }
        }
        // forward substitution with the finished columns
#pragma unroll 1
        for (int k = 0; k < j; k++) {
            const double u1 = TL(c1, k), ur = TL(cr, k), ui = TL(ci, k);
            const double *l1 = g1 + k * N * 32;
            const double2 *l2 = g2 + k * N * 32;
#pragma unroll 4
            for (int i = k + 1; i < N; i++) {
                const double a = TL(l1, i);
                const double2 b = TL(l2, i);
                TL(c1, i) = fma(-a, u1, TL(c1, i));
                TL(cr, i) = fma(-b.x, ur, fma(b.y, ui, TL(cr, i)));
                TL(ci, i) = fma(-b.x, ui, fma(-b.y, ur, TL(ci, i)));
            }
        }
        // pivots
        double best1 = -1.0, best2 = -1.0;
        int p1 = j, p2 = j;
#pragma unroll 1
        for (int i = j; i < N; i++) {
            const double v1 = fabs(TL(c1, i)), v2 = fabs(TL(cr, i)) + fabs(TL(ci, i));
            if (v1 > best1) { best1 = v1; p1 = i; }
            if (v2 > best2) { best2 = v2; p2 = i; }
        }
        if (!ier && (bad || !(best1 > 0.0) || !isfinite(best1) || !(best2 > 0.0) || !isfinite(best2))) ier = j + 1;
        ip1 |= (u64)p1 << (4 * j);
        ip2 |= (u64)p2 << (4 * j);
        if (p1 != j) {
            const double t = TL(c1, j); TL(c1, j) = TL(c1, p1); TL(c1, p1) = t;
#pragma unroll 1
            for (int k = 0; k < j; k++) { const double s = TL(g1, k * N + j); TL(g1, k * N + j) = TL(g1, k * N + p1); TL(g1, k * N + p1) = s; }
        }
        if (p2 != j) {
            const double t = TL(cr, j), s = TL(ci, j);
            TL(cr, j) = TL(cr, p2); TL(ci, j) = TL(ci, p2);
            TL(cr, p2) = t; TL(ci, p2) = s;
#pragma unroll 1
            for (int k = 0; k < j; k++) { const double2 w = TL(g2, k * N + j); TL(g2, k * N + j) = TL(g2, k * N + p2); TL(g2, k * N + p2) = w; }
        }
        const double r1 = rcp_f(TL(c1, j));
        const double pr = TL(cr, j), pi = TL(ci, j);
        const double den = rcp_f(pr * pr + pi * pi);
        const double qr = pr * den, qi = -pi * den;            // 1 / pivot
        double *o1 = g1 + j * N * 32;
        double2 *o2 = g2 + j * N * 32;
#pragma unroll 4
        for (int i = 0; i < N; i++) {
            double a = TL(c1, i), br = TL(cr, i), bi = TL(ci, i);
            if (i > j) {
                a *= r1;
                const double tr = br * qr - bi * qi, ti = br * qi + bi * qr;
                br = tr; bi = ti;
            } else if (i == j) {
                a = r1; br = qr; bi = qi;
            }
            TL(o1, i) = a;
            TL(o2, i) = make_double2(br, bi);
        }
    }
    ip1_out = ip1;
    ip2_out = ip2;
    return ier;
}

__device__ __forceinline__ void apply_perm(double *b, int N, u64 ip)
{
#pragma unroll 1
    for (int k = 0; k < N; k++) {
        const int p = (int)(ip >> (4 * k)) & 15;
        if (p != k) { const double t = TL(b, k); TL(b, k) = TL(b, p); TL(b, p) = t; }
    }
}

// E1 x = b in place (b lane-private in shared memory)
static __device__ __noinline__ void solve_real(const double *g1, double *b, int N, u64 ip)
{
    apply_perm(b, N, ip);
#pragma unroll 1
    for (int i = 1; i < N; i++) {
        double s = TL(b, i);
#pragma unroll 4
        for (int k = 0; k < i; k++) s = fma(-TL(g1, k * N + i), TL(b, k), s);
        TL(b, i) = s;
    }
#pragma unroll 1
    for (int i = N - 1; i >= 0; i--) {
        double s = TL(b, i);
#pragma unroll 4
        for (int j = i + 1; j < N; j++) s = fma(-TL(g1, j * N + i), TL(b, j), s);
        TL(b, i) = s * TL(g1, i * N + i);
    }
}

// E1 x1 = b1 and E2 (x2 + i x3) = b2 + i b3 in place, one loop nest (three independent dependency chains)
static __device__ __noinline__ void solve3(const double *g1, const double2 *g2, double *b1, double *b2, double *b3, int N, u64 ip1, u64 ip2)
{
    apply_perm(b1, N, ip1);
#pragma unroll 1
    for (int k = 0; k < N; k++) {
        const int p = (int)(ip2 >> (4 * k)) & 15;
        if (p != k) {
            const double t = TL(b2, k), s = TL(b3, k);
            TL(b2, k) = TL(b2, p); TL(b3, k) = TL(b3, p);
            TL(b2, p) = t; TL(b3, p) = s;
        }
    }
#pragma unroll 1
    for (int i = 1; i < N; i++) {
        double s1 = TL(b1, i), sr = TL(b2, i), si = TL(b3, i);
#pragma unroll 4
        for (int k = 0; k < i; k++) {
            const double a = TL(g1, k * N + i);
            const double2 c = TL(g2, k * N + i);
            const double x1 = TL(b1, k), xr = TL(b2, k), xi = TL(b3, k);
            s1 = fma(-a, x1, s1);
            sr = fma(-c.x, xr, fma(c.y, xi, sr));
            si = fma(-c.x, xi, fma(-c.y, xr, si));
        }
        TL(b1, i) = s1; TL(b2, i) = sr; TL(b3, i) = si;
    }
#pragma unroll 1
    for (int i = N - 1; i >= 0; i--) {
        double s1 = TL(b1, i), sr = TL(b2, i), si = TL(b3, i);
#pragma unroll 4
        for (int j = i + 1; j < N; j++) {
            const double a = TL(g1, j * N + i);
            const double2 c = TL(g2, j * N + i);
            const double x1 = TL(b1, j), xr = TL(b2, j), xi = TL(b3, j);
            s1 = fma(-a, x1, s1);
            sr = fma(-c.x, xr, fma(c.y, xi, sr));
            si = fma(-c.x, xi, fma(-c.y, xr, si));
        }
        const double2 d = TL(g2, i * N + i);
        TL(b1, i) = s1 * TL(g1, i * N + i);
        TL(b2, i) = sr * d.x - si * d.y;
        TL(b3, i) = sr * d.y + si * d.x;
    }
}

// ------------------------------------------------------------------------------------------------ the same for a
// compile-time N: the column of the factorisation and the right-hand sides of the solves live in REGISTERS (static
// indices only), every global load has a compile-time offset and no dependence on the arithmetic (the compiler issues
// them far ahead of their use: the loops of the runtime-N routines above stall on L2 latency), and the row
// interchanges are carried as a permutation packed four bits per position (perm: position -> original row), applied
// when a column of J is LOADED, so that finished columns never have to be permuted in registers.
__device__ __forceinline__ u64 perm_swap(u64 perm, int a, int b)
{
    const u64 x = ((perm >> (4 * a)) ^ (perm >> (4 * b))) & 15ull;
    return perm ^ (x << (4 * a)) ^ (x << (4 * b));
}

template <int N>
__device__ __noinline__ int lu_pair_t(const double *gJ, double *g1, double2 *g2, double *col, double fac1, double alphn,
                                      double betan, u64 &perm1_out, u64 &perm2_out, bool keep)
{
    const u64 pol = l2_policy(keep), pol_j = l2_policy(false);
    double *s1 = col, *sr = col + N * 32, *si = col + 2 * N * 32;
    u64 perm1 = 0xFEDCBA9876543210ull, perm2 = 0xFEDCBA9876543210ull;
    int ier = 0;
#pragma unroll 1
    for (int j = 0; j < N; j++) {
        double c1[N], cr[N], ci[N];
        bool bad = false;
#pragma unroll
        for (int i = 0; i < N; i++) {
            const int r1 = (int)(perm1 >> (4 * i)) & 15, r2 = (int)(perm2 >> (4 * i)) & 15;
            const double v1 = -TLP(gJ, r1 * N + j, pol_j), v2 = -TLP(gJ, r2 * N + j, pol_j);
            bad |= !isfinite(v1);
            c1[i] = r1 == j ? v1 + fac1 : v1;
            cr[i] = r2 == j ? v2 + alphn : v2;
            ci[i] = r2 == j ? betan : 0.0;
        }
#pragma unroll
        for (int k = 0; k < N - 1; k++) {
            if (k < j) {
                const double u1 = c1[k], ur = cr[k], ui = ci[k];
#pragma unroll
                for (int i = k + 1; i < N; i++) {
                    const double a = TLP(g1, k * N + i, pol);
                    const double2 b = TLP(g2, k * N + i, pol);
                    c1[i] = fma(-a, u1, c1[i]);
                    cr[i] = fma(-b.x, ur, fma(b.y, ui, cr[i]));
                    ci[i] = fma(-b.x, ui, fma(-b.y, ur, ci[i]));
                }
            }
        }
        double best1 = -1.0, best2 = -1.0;
        int p1 = j, p2 = j;
#pragma unroll
        for (int i = 0; i < N; i++) {
            const double v1 = fabs(c1[i]), v2 = fabs(cr[i]) + fabs(ci[i]);
            TL(s1, i) = c1[i]; TL(sr, i) = cr[i]; TL(si, i) = ci[i];
            if (i >= j && v1 > best1) { best1 = v1; p1 = i; }
            if (i >= j && v2 > best2) { best2 = v2; p2 = i; }
        }
        if (!ier && (bad || !(best1 > 0.0) || !isfinite(best1) || !(best2 > 0.0) || !isfinite(best2))) ier = j + 1;
        if (p1 != j) {
            const double t = TL(s1, j); TL(s1, j) = TL(s1, p1); TL(s1, p1) = t;
            perm1 = perm_swap(perm1, j, p1);
#pragma unroll 2
            for (int k = 0; k < j; k++) { const double s = TLP(g1, k * N + j, pol); stp(&TL(g1, k * N + j), TLP(g1, k * N + p1, pol), pol); stp(&TL(g1, k * N + p1), s, pol); }
        }
        if (p2 != j) {
            const double t = TL(sr, j), s = TL(si, j);
            TL(sr, j) = TL(sr, p2); TL(si, j) = TL(si, p2);
            TL(sr, p2) = t; TL(si, p2) = s;
            perm2 = perm_swap(perm2, j, p2);
#pragma unroll 2
            for (int k = 0; k < j; k++) { const double2 w = TLP(g2, k * N + j, pol); stp(&TL(g2, k * N + j), TLP(g2, k * N + p2, pol), pol); stp(&TL(g2, k * N + p2), w, pol); }
        }
        const double r1 = rcp_f(TL(s1, j));
        const double pr = TL(sr, j), pi = TL(si, j);
        const double den = rcp_f(pr * pr + pi * pi);
        const double qr = pr * den, qi = -pi * den;            // 1 / pivot
        double *o1 = g1 + j * N * 32;
        double2 *o2 = g2 + j * N * 32;
#pragma unroll
        for (int i = 0; i < N; i++) {
            double a = TL(s1, i), br = TL(sr, i), bi = TL(si, i);
            if (i > j) {
                a *= r1;
                const double tr = br * qr - bi * qi, ti = br * qi + bi * qr;
                br = tr; bi = ti;
            } else if (i == j) {
                a = r1; br = qr; bi = qi;
            }
            stp(&TL(o1, i), a, pol);
            stp(&TL(o2, i), make_double2(br, bi), pol);
        }
    }
    perm1_out = perm1;
    perm2_out = perm2;
    return ier;
}

// E1 x = b; b is read from `b` through the permutation and x written back to `b` (lane-private, shared memory)
template <int N>
__device__ __noinline__ void solve_real_t(const double *g1, double *b, u64 perm, bool keep)
{
    const u64 pol = l2_policy(keep);
    double x[N];
#pragma unroll
    for (int i = 0; i < N; i++) x[i] = TL(b, (int)(perm >> (4 * i)) & 15);
#pragma unroll
    for (int i = 1; i < N; i++)
#pragma unroll
        for (int k = 0; k < i; k++) x[i] = fma(-TLP(g1, k * N + i, pol), x[k], x[i]);
#pragma unroll
    for (int i = N - 1; i >= 0; i--) {
#pragma unroll
        for (int j = i + 1; j < N; j++) x[i] = fma(-TLP(g1, j * N + i, pol), x[j], x[i]);
        x[i] *= TLP(g1, i * N + i, pol);
    }
#pragma unroll
    for (int i = 0; i < N; i++) TL(b, i) = x[i];
}

// E1 x1 = b1 and E2 (x2 + i x3) = b2 + i b3, right-hand sides and solutions in z = [b1 | b2 | b3] (shared memory)
template <int N>
__device__ __noinline__ void solve3_t(const double *g1, const double2 *g2, double *z, u64 perm1, u64 perm2, bool keep)
{
    const u64 pol = l2_policy(keep);
    double x1[N], xr[N], xi[N];
#pragma unroll
    for (int i = 0; i < N; i++) {
        const int r1 = (int)(perm1 >> (4 * i)) & 15, r2 = (int)(perm2 >> (4 * i)) & 15;
        x1[i] = TL(z, r1); xr[i] = TL(z, N + r2); xi[i] = TL(z, 2 * N + r2);
    }
#pragma unroll
    for (int i = 1; i < N; i++)
#pragma unroll
        for (int k = 0; k < i; k++) {
            const double a = TLP(g1, k * N + i, pol);
            const double2 c = TLP(g2, k * N + i, pol);
            x1[i] = fma(-a, x1[k], x1[i]);
            xr[i] = fma(-c.x, xr[k], fma(c.y, xi[k], xr[i]));
            xi[i] = fma(-c.x, xi[k], fma(-c.y, xr[k], xi[i]));
        }
#pragma unroll
    for (int i = N - 1; i >= 0; i--) {
#pragma unroll
        for (int j = i + 1; j < N; j++) {
            const double a = TLP(g1, j * N + i, pol);
            const double2 c = TLP(g2, j * N + i, pol);
            x1[i] = fma(-a, x1[j], x1[i]);
            xr[i] = fma(-c.x, xr[j], fma(c.y, xi[j], xr[i]));
            xi[i] = fma(-c.x, xi[j], fma(-c.y, xr[j], xi[i]));
        }
        const double2 d = TLP(g2, i * N + i, pol);
        x1[i] *= TLP(g1, i * N + i, pol);
        const double tr = xr[i] * d.x - xi[i] * d.y, ti = xr[i] * d.y + xi[i] * d.x;
        xr[i] = tr; xi[i] = ti;
    }
#pragma unroll
    for (int i = 0; i < N; i++) { TL(z, i) = x1[i]; TL(z, N + i) = xr[i]; TL(z, 2 * N + i) = xi[i]; }
}

}  // namespace tps
}  // namespace chem

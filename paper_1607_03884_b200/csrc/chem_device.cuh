// chem_device.cuh -- group-cooperative device routines: thermo, species rates, source term,
// analytical Jacobian, dense LU / solves (real and complex), and the Radau IIA step engine.
//
// A "group" is G threads that own ONE thermochemical state: a warp (G = 32) for small mechanisms,
// a whole CTA (G = 128) for GRI-sized ones.  Control flow is uniform inside a group, so the
// intra-warp divergence the paper names as its first limiter does not occur;
// all per-state data (Jacobian, LU factors, stage vectors) lives in shared memory, which removes the
// second limiter (L182: "storage of the Jacobian matrix and/or factorized forms ... overwhelm the
// registers and L1").  See DESIGN.md for the readings R1..R12 cited below.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

#include "chem_common.cuh"

namespace chem {

// ---------------------------------------------------------------------------------------------
template <int G>
struct Grp {
    static constexpr int NW = G / 32;
    __device__ static __forceinline__ int lane() { return G == 32 ? (threadIdx.x & 31) : (int)threadIdx.x; }
    __device__ static __forceinline__ int wlane() { return threadIdx.x & 31; }
    __device__ static __forceinline__ int warp() { return G == 32 ? 0 : (int)(threadIdx.x >> 5); }
    __device__ static __forceinline__ void sync()
    {
        if (G == 32) __syncwarp(); else __syncthreads();
    }
    // all-reduce of two sums; every thread of the group gets bitwise the same result.
    // `red` = shared scratch of 2*NW doubles (unused for G == 32).
    __device__ static __forceinline__ void sum2(double &a, double &b, double *red)
    {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            a += __shfl_xor_sync(0xffffffffu, a, o);
            b += __shfl_xor_sync(0xffffffffu, b, o);
        }
        if (G > 32) {
            __syncthreads();
            if (wlane() == 0) { red[2 * warp()] = a; red[2 * warp() + 1] = b; }
            __syncthreads();
            a = 0.0; b = 0.0;
#pragma unroll
            for (int w = 0; w < NW; w++) { a += red[2 * w]; b += red[2 * w + 1]; }
        }
    }
    __device__ static __forceinline__ int any(int p, double *red)
    {
        if (G == 32) return __any_sync(0xffffffffu, p);
        return __syncthreads_or(p);
    }
};

// Rebase a generic pointer that is known to point into this CTA's dynamic shared memory on the shared window, so that
// the compiler emits LDS / STS instead of generic LD / ST inside out-of-line routines (where it cannot see the origin
// of pointer arguments and struct members).
template <typename T>
__device__ __forceinline__ T *shp(T *p)
{
    extern __shared__ double chem_smem_window_[];
    const size_t off = __cvta_generic_to_shared(p) - __cvta_generic_to_shared(chem_smem_window_);
    return reinterpret_cast<T *>(reinterpret_cast<char *>(chem_smem_window_) + off);
}

__device__ __forceinline__ double powi(double c, int nu)
{
    return nu == 0 ? 1.0 : (nu == 1 ? c : (nu == 2 ? c * c : c * c * c));
}
__device__ __forceinline__ double dpowi(double c, int nu)  // d/dc c^nu
{
    return nu == 0 ? 0.0 : (nu == 1 ? 1.0 : (nu == 2 ? 2.0 * c : 3.0 * c * c));
}

// Chemistry scratch of one group (shared memory).
struct ChemScratch {
    double *C, *g, *hRT, *cpR, *dcpR, *wdot;  // [n_sp]
    double *q;                                // [n_rx]
    double *dq;                               // [6][n_rx]   (Jacobian only)
    double *dqdT, *tb;                        // [n_rx]      (Jacobian only)
    double *red;                              // [2*NW]
    double *jpool;                            // private rows of the balanced Jacobian gather (dead matrix storage)
};

__device__ __forceinline__ ChemScratch shp(const ChemScratch &g)
{
    ChemScratch s;
    s.C = shp(g.C); s.g = shp(g.g); s.hRT = shp(g.hRT); s.cpR = shp(g.cpR); s.dcpR = shp(g.dcpR); s.wdot = shp(g.wdot);
    s.q = shp(g.q); s.dq = shp(g.dq); s.dqdT = shp(g.dqdT); s.tb = shp(g.tb); s.red = shp(g.red); s.jpool = g.jpool ? shp(g.jpool) : nullptr;
    return s;
}

// Mixture state derived from ys = (T, Y_1..Y_{N-1}): fills C, g = h/RT - s/R, hRT, cpR (and dcpR).
// DESIGN.md R1 (state, closure, ideal gas) and R2 (NASA-7).
template <int G, bool JAC>
__device__ __forceinline__ void front_end(const Tables &t, const ChemScratch &s, double P, const double *ys, double &T,
                                          double &rho, double &Wbar)
{
    const int N = t.n_sp;
    const int lane = Grp<G>::lane();
    T = ys[0];
    double sY = 0.0, sYW = 0.0;
    for (int k = lane; k < N - 1; k += G) {
        const double Yk = ys[k + 1];
        sY += Yk;
        sYW += Yk * __ldg(&t.invW[k]);
    }
    Grp<G>::sum2(sY, sYW, s.red);
    const double YN = 1.0 - sY;
    sYW += YN * __ldg(&t.invW[N - 1]);
    Wbar = 1.0 / sYW;
    rho = P * Wbar / (kRerg * T);
    const double lnT = log(T);
    const double invT = 1.0 / T;
    for (int k = lane; k < N; k += G) {
        const double Yk = (k < N - 1) ? ys[k + 1] : YN;
        s.C[k] = rho * Yk * __ldg(&t.invW[k]);
        const double *a = (T <= __ldg(&t.tmid[k])) ? t.nasa_lo : t.nasa_hi;
        const double a0 = __ldg(&a[k]), a1 = __ldg(&a[N + k]), a2 = __ldg(&a[2 * N + k]), a3 = __ldg(&a[3 * N + k]);
        const double a4 = __ldg(&a[4 * N + k]), a5 = __ldg(&a[5 * N + k]), a6 = __ldg(&a[6 * N + k]);
        const double cp = a0 + T * (a1 + T * (a2 + T * (a3 + T * a4)));
        const double h = a0 + T * (a1 * 0.5 + T * (a2 * (1.0 / 3.0) + T * (a3 * 0.25 + T * (a4 * 0.2)))) + a5 * invT;
        const double sR = a0 * lnT + T * (a1 + T * (a2 * 0.5 + T * (a3 * (1.0 / 3.0) + T * (a4 * 0.25)))) + a6;
        s.cpR[k] = cp;
        s.hRT[k] = h;
        s.g[k] = h - sR;
        if (JAC) s.dcpR[k] = a1 + T * (2.0 * a2 + T * (3.0 * a3 + T * (4.0 * a4)));
    }
    Grp<G>::sync();
}

// Rate of progress of reaction i (R3 mass action + Arrhenius + Kc, R4 third body, R5 falloff/Troe).
// With JAC also the partial derivatives at constant C (dq/dT), per slot (dq/dC_slot) and through [M] (tb).
template <bool JAC>
__device__ __forceinline__ double reaction(const Tables &t, int i, double T, double lnT, double invT, double lnPRT,
                                           double Ctot, const ChemScratch &s)
{
    const int NR = t.n_rx;
    const double b = __ldg(&t.b[i]), Ta = __ldg(&t.Ta[i]);
    const double lnkf = __ldg(&t.lnA[i]) + b * lnT - Ta * invT;
    double dG = 0.0, dH = 0.0;
    double pw[kSlots], cs[kSlots];
    int nus[kSlots];
#pragma unroll
    for (int sl = 0; sl < kSlots; sl++) {
        const int sp = __ldg(&t.slot_sp[sl * NR + i]);
        const int nu = __ldg(&t.slot_nu[sl * NR + i]);
        const double c = s.C[sp];
        const double sgn = (sl < 3) ? -(double)nu : (double)nu;
        dG += sgn * s.g[sp];
        if (JAC) dH += sgn * s.hRT[sp];
        pw[sl] = powi(c, nu);
        cs[sl] = c;
        nus[sl] = nu;
    }
    const double dnu = __ldg(&t.dnu[i]);
    const double kf = exp(lnkf);
    const double kr = exp(lnkf - (dnu * lnPRT - dG));   // kf / Kc
    const double Rf = kf * (pw[0] * pw[1] * pw[2]);
    const double Rr = kr * (pw[3] * pw[4] * pw[5]);
    const double rnet = Rf - Rr;
    const int type = __ldg(&t.rtype[i]);
    double c = 1.0, dc_dT = 0.0, dc_dM = 0.0;
    const double dlnkf = (b + Ta * invT) * invT;
    if (type != 0) {
        double M = Ctot;
        for (int p = __ldg(&t.eff_ptr[i]); p < __ldg(&t.eff_ptr[i + 1]); p++)
            M += __ldg(&t.eff_dv[p]) * s.C[__ldg(&t.eff_sp[p])];
        if (type == 1) {
            c = M;
            dc_dM = 1.0;
        } else {
            const double b0 = __ldg(&t.b0[i]), Ta0 = __ldg(&t.Ta0[i]);
            const double k0_over_kinf = exp(__ldg(&t.lnA0[i]) + b0 * lnT - Ta0 * invT - lnkf);
            const double Pr = k0_over_kinf * M;
            const double dlnPr_dT = (b0 + Ta0 * invT) * invT - dlnkf;
            double F = 1.0, dF_dT = 0.0, dF_dPr = 0.0;
            if (type == 3) {
                const double al = __ldg(&t.troe[i]), T3 = __ldg(&t.troe[NR + i]);
                const double T1 = __ldg(&t.troe[2 * NR + i]), T2 = __ldg(&t.troe[3 * NR + i]);
                const double e3 = (1.0 - al) * exp(-T / T3), e1 = al * exp(-T / T1), e2 = exp(-T2 * invT);
                const double Fc = e3 + e1 + e2;
                const double L = log10(Fc);
                const double cc = -0.4 - 0.67 * L, nn = 0.75 - 1.27 * L;
                const double At = log10(Pr) + cc;
                const double Bt = nn - 0.14 * At;
                const double x = At / Bt;
                const double den = 1.0 + x * x;
                F = exp10(L / den);
                if (JAC) {
                    const double ln10 = 2.302585092994045684;
                    const double dFc = -e3 / T3 - e1 / T1 + e2 * T2 * invT * invT;
                    const double dL = dFc / (Fc * ln10);
                    const double dA_T = dlnPr_dT / ln10 - 0.67 * dL;
                    const double dB_T = -1.27 * dL - 0.14 * dA_T;
                    const double dx_T = (dA_T * Bt - At * dB_T) / (Bt * Bt);
                    const double dA_P = 1.0 / (Pr * ln10);
                    const double dx_P = dA_P * (Bt + 0.14 * At) / (Bt * Bt);
                    const double w = -L * 2.0 * x / (den * den);
                    dF_dT = F * ln10 * (dL / den + w * dx_T);
                    dF_dPr = F * ln10 * w * dx_P;
                }
            }
            const double op = 1.0 / (1.0 + Pr);
            c = Pr * op * F;
            if (JAC) {
                dc_dT = Pr * dlnPr_dT * op * op * F + Pr * op * dF_dT;
                dc_dM = (op * op * F + Pr * op * dF_dPr) * k0_over_kinf;
            }
        }
    }
    const double q = c * rnet;
    if (JAC) {
        // van 't Hoff: d ln kr/dT = d ln kf/dT - (sum nu h/RT - dnu)/T
        const double dlnkr = dlnkf - (dH - dnu) * invT;
        s.dqdT[i] = dc_dT * rnet + c * (Rf * dlnkf - Rr * dlnkr);
        s.tb[i] = dc_dM * rnet;
        const double ckf = c * kf, ckr = c * kr;
        s.dq[0 * NR + i] = ckf * dpowi(cs[0], nus[0]) * pw[1] * pw[2];
        s.dq[1 * NR + i] = ckf * dpowi(cs[1], nus[1]) * pw[0] * pw[2];
        s.dq[2 * NR + i] = ckf * dpowi(cs[2], nus[2]) * pw[0] * pw[1];
        s.dq[3 * NR + i] = -ckr * dpowi(cs[3], nus[3]) * pw[4] * pw[5];
        s.dq[4 * NR + i] = -ckr * dpowi(cs[4], nus[4]) * pw[3] * pw[5];
        s.dq[5 * NR + i] = -ckr * dpowi(cs[5], nus[5]) * pw[3] * pw[4];
    }
    return q;
}

// Source term f(T, Y; P) of one state (R1): f[0] = dT/dt, f[k+1] = dY_k/dt.  ys, f: shared, length N.
template <int G>
__device__ __noinline__ void rhs(const Tables &tg, const ChemScratch &sg, double P, const double *ys, double *f)
{
    const ChemScratch s = shp(sg);     // shared-memory scratch: LDS / STS instead of generic accesses
    ys = shp(ys); f = shp(f);
    const Tables &t = *shp(&tg);
    const int N = t.n_sp, NR = t.n_rx;
    const int lane = Grp<G>::lane();
    double T, rho, Wbar;
    front_end<G, false>(t, s, P, ys, T, rho, Wbar);
    const double lnT = log(T), invT = 1.0 / T;
    const double Ctot = P / (kRerg * T);
    const double lnPRT = log(kPatm / (kRerg * T));
    for (int i = lane; i < NR; i += (lane < t.n_solo ? NR : G - t.n_solo)) s.q[i] = reaction<false>(t, i, T, lnT, invT, lnPRT, Ctot, s);
    Grp<G>::sync();
    double hw = 0.0, ccp = 0.0;
    for (int k = lane; k < N; k += G) {
        double w = 0.0;
        for (int p = __ldg(&t.inc_ptr[k]); p < __ldg(&t.inc_ptr[k + 1]); p++)
            w += __ldg(&t.inc_nu[p]) * s.q[__ldg(&t.inc_rx[p])];
        hw += s.hRT[k] * w;
        ccp += s.C[k] * s.cpR[k];
        if (k < N - 1) f[k + 1] = __ldg(&t.W[k]) * w / rho;
    }
    Grp<G>::sum2(hw, ccp, s.red);
    if (lane == 0) f[0] = -T * hw / ccp;
    Grp<G>::sync();
}

// Analytical Jacobian (R6), Jm: shared N x N row-major, Jm[i*N+j] = d f_i / d y_j.
// Uses that at constant (T, P) the total concentration is independent of Y, so the unit part of the
// third-body efficiencies only enters d/dT.
template <int G>
__device__ __noinline__ void jacobian(const Tables &tg, const ChemScratch &sg, double P, const double *ys, double *Jm)
{
    const ChemScratch s = shp(sg);     // shared-memory scratch: LDS / STS instead of generic accesses
    ys = shp(ys); Jm = shp(Jm);
    const Tables &t = *shp(&tg);
    const int N = t.n_sp, NR = t.n_rx;
    const int lane = Grp<G>::lane();
    double T, rho, Wbar;
    front_end<G, true>(t, s, P, ys, T, rho, Wbar);
    const double lnT = log(T), invT = 1.0 / T;
    const double Ctot = P / (kRerg * T);
    const double lnPRT = log(kPatm / (kRerg * T));
    for (int i = lane; i < NR; i += (lane < t.n_solo ? NR : G - t.n_solo)) s.q[i] = reaction<true>(t, i, T, lnT, invT, lnPRT, Ctot, s);
    Grp<G>::sync();
    const double invWN = __ldg(&t.invW[N - 1]);
    // rows: species k -> Dw[k][j] = d wdot_k / d y_j, stored in Jm row k.
    // Balanced gather (CTA groups): a few radicals take part in a third of the reactions, and one thread per species
    // left the group waiting for the longest incidence list.  Species k gets 2^m adjacent threads (schedule from the
    // mechanism compiler), each accumulates its share of the list in a private row of N + 3 doubles (row, wdot,
    // d wdot/dT at constant C, third-body sum) in matrix storage that is dead while the Jacobian is evaluated, and the
    // shares are added in a fixed order (deterministic).  One packed record per incidence: one trip to L2.
    const bool balanced = G == 128 && t.gatj_T > 0 && s.jpool != nullptr;
    if (balanced) {
        const int RS = N + 3;
        int4 g = make_int4(-1, 0, 0, 0);
        if (lane < t.gatj_T) g = __ldg(t.gatj + lane);
        double *row = s.jpool + lane * RS;
        if (g.x >= 0) {
            for (int l = 0; l < RS; l++) row[l] = 0.0;
            double wd = 0.0, dwT = 0.0, u = 0.0;
#pragma unroll 2
            for (int p = g.y; p < g.z; p++) {
                const int4 e0 = __ldg(t.jinc + 2 * p), e1 = __ldg(t.jinc + 2 * p + 1);
                const int i = e0.x;
                const double nu = (double)e0.y;
                wd += nu * s.q[i];
                dwT += nu * s.dqdT[i];
                row[e0.z & 255] += nu * s.dq[i];
                row[(e0.z >> 8) & 255] += nu * s.dq[NR + i];
                row[(e0.z >> 16) & 255] += nu * s.dq[2 * NR + i];
                row[e0.w & 255] += nu * s.dq[3 * NR + i];
                row[(e0.w >> 8) & 255] += nu * s.dq[4 * NR + i];
                row[(e0.w >> 16) & 255] += nu * s.dq[5 * NR + i];
                if (e1.z) {
                    const double v = nu * s.tb[i];
                    u += v;
                    for (int pe = e1.x; pe < e1.y; pe++) row[__ldg(&t.eff_sp[pe])] += v * __ldg(&t.eff_dv[pe]);
                }
            }
            row[N] = wd; row[N + 1] = dwT; row[N + 2] = u;
        }
        Grp<G>::sync();
        if (g.x >= 0) {
            const int c = 1 << g.w, qi = lane & (c - 1);      // groups are aligned to their (power of two) size
            const double *first = s.jpool + (lane - qi) * RS;
            for (int l = qi; l < RS; l += c) {
                double sum = 0.0;
                for (int m = 0; m < c; m++) sum += first[m * RS + l];
                if (l < N) Jm[g.x * N + l] = sum;
                else if (l == N) s.wdot[g.x] = sum;
                else s.dq[(l - N - 1) * N + g.x] = sum;       // dq is dead by now: [0,N) d wdot/dT, [N,2N) third-body sums
            }
        }
        Grp<G>::sync();
    }
    double hw = 0.0, ccp = 0.0, cpw = 0.0, cdcp = 0.0;
    for (int k = lane; k < N; k += G) {
        double *row = Jm + k * N;
        double wd = 0.0, dwT = 0.0, u = 0.0;
        if (balanced) {
            wd = s.wdot[k]; dwT = s.dq[k]; u = s.dq[N + k];
        } else {
            for (int l = 0; l < N; l++) row[l] = 0.0;
            for (int p = __ldg(&t.inc_ptr[k]); p < __ldg(&t.inc_ptr[k + 1]); p++) {
                const int i = __ldg(&t.inc_rx[p]);
                const double nu = __ldg(&t.inc_nu[p]);
                wd += nu * s.q[i];
                dwT += nu * s.dqdT[i];
#pragma unroll
                for (int sl = 0; sl < kSlots; sl++) row[__ldg(&t.slot_sp[sl * NR + i])] += nu * s.dq[sl * NR + i];
                if (__ldg(&t.rtype[i]) != 0) {
                    const double v = nu * s.tb[i];
                    u += v;
                    for (int pe = __ldg(&t.eff_ptr[i]); pe < __ldg(&t.eff_ptr[i + 1]); pe++)
                        row[__ldg(&t.eff_sp[pe])] += v * __ldg(&t.eff_dv[pe]);
                }
            }
        }
        double GC = 0.0;
        for (int l = 0; l < N; l++) GC += row[l] * s.C[l];
        const double GN = row[N - 1] * invWN;
        for (int j = N - 1; j >= 1; j--) {
            const double dj = __ldg(&t.invW[j - 1]) - invWN;
            row[j] = -Wbar * dj * GC + rho * (row[j - 1] * __ldg(&t.invW[j - 1]) - GN);
        }
        row[0] = dwT - (GC + u * Ctot) * invT;
        s.wdot[k] = wd;
        hw += s.hRT[k] * wd;
        ccp += s.C[k] * s.cpR[k];
        cpw += s.cpR[k] * wd;
        cdcp += s.C[k] * s.dcpR[k];
    }
    Grp<G>::sum2(hw, ccp, s.red);
    Grp<G>::sum2(cpw, cdcp, s.red);
    Grp<G>::sync();
    const double Tdot = -T * hw / ccp;
    // columns: assemble the rows of J in place (row k+1 <- species k, descending; row 0 <- temperature)
    for (int j = lane; j < N; j += G) {
        double S = 0.0;
        for (int k = 0; k < N; k++) S += s.hRT[k] * Jm[k * N + j];
        double dlnrho, drcp;   // d ln rho / d y_j ; d(sum C cpR) / d y_j
        if (j == 0) {
            dlnrho = -invT;
            drcp = -ccp * invT + cdcp;
        } else {
            const double dj = __ldg(&t.invW[j - 1]) - invWN;
            dlnrho = -Wbar * dj;
            drcp = -Wbar * dj * ccp + rho * (s.cpR[j - 1] * __ldg(&t.invW[j - 1]) - s.cpR[N - 1] * invWN);
        }
        for (int k = N - 2; k >= 0; k--) {
            const double Wk = __ldg(&t.W[k]);
            Jm[(k + 1) * N + j] = Wk / rho * Jm[k * N + j] - Wk * s.wdot[k] / rho * dlnrho;
        }
        Jm[j] = -(T * S + (j == 0 ? cpw : 0.0)) / ccp - Tdot * drcp / ccp;
    }
    Grp<G>::sync();
}

// ------------------------------------------------------------------------------------- dense LU
// Column-major N x N in shared memory: A[i + j*N].  Partial pivoting with full-row interchanges
// (LAPACK convention), first maximum wins ties.  Returns 0 or k+1 (zero / non-finite pivot column).
// "specialized implementations of ... LU factorization of the Jacobian".
template <int G>
__device__ __noinline__ int lu_real(int N, double *A, int *ip)
{
    const int lane = Grp<G>::lane(), wl = Grp<G>::wlane(), wp = Grp<G>::warp();
    for (int k = 0; k < N; k++) {
        double best = -1.0;
        int bi = k;
        for (int i = k + wl; i < N; i += 32) {
            const double v = fabs(A[i + k * N]);
            if (v > best) { best = v; bi = i; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, best, o);
            const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (ov > best || (ov == best && oi < bi)) { best = ov; bi = oi; }
        }
        if (lane == 0) ip[k] = bi;
        if (!(best > 0.0) || !isfinite(best)) return k + 1;
        Grp<G>::sync();   // every warp has read column k before rows move
        if (bi != k)
            for (int j = lane; j < N; j += G) {
                const double a = A[k + j * N];
                A[k + j * N] = A[bi + j * N];
                A[bi + j * N] = a;
            }
        Grp<G>::sync();
        const double piv = A[k + k * N];
        Grp<G>::sync();
        for (int i = k + 1 + lane; i < N; i += G) A[i + k * N] /= piv;
        Grp<G>::sync();
        for (int j = k + 1 + wp; j < N; j += Grp<G>::NW) {
            const double u = A[k + j * N];
            for (int i = k + 1 + wl; i < N; i += 32) A[i + j * N] -= A[i + k * N] * u;
        }
        Grp<G>::sync();
    }
    return 0;
}

// Complex version on split planes (Ar, Ai); pivot magnitude |re| + |im| (R10).
template <int G>
__device__ __noinline__ int lu_complex(int N, double *Ar, double *Ai, int *ip)
{
    const int lane = Grp<G>::lane(), wl = Grp<G>::wlane(), wp = Grp<G>::warp();
    for (int k = 0; k < N; k++) {
        double best = -1.0;
        int bi = k;
        for (int i = k + wl; i < N; i += 32) {
            const double v = fabs(Ar[i + k * N]) + fabs(Ai[i + k * N]);
            if (v > best) { best = v; bi = i; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, best, o);
            const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (ov > best || (ov == best && oi < bi)) { best = ov; bi = oi; }
        }
        if (lane == 0) ip[k] = bi;
        if (!(best > 0.0) || !isfinite(best)) return k + 1;
        Grp<G>::sync();
        if (bi != k)
            for (int j = lane; j < N; j += G) {
                double a = Ar[k + j * N];
                Ar[k + j * N] = Ar[bi + j * N];
                Ar[bi + j * N] = a;
                a = Ai[k + j * N];
                Ai[k + j * N] = Ai[bi + j * N];
                Ai[bi + j * N] = a;
            }
        Grp<G>::sync();
        const double pr = Ar[k + k * N], pi = Ai[k + k * N];
        Grp<G>::sync();
        // l = a / p = a conj(p) / |p|^2
        const double den = 1.0 / (pr * pr + pi * pi);
        for (int i = k + 1 + lane; i < N; i += G) {
            const double ar = Ar[i + k * N], ai = Ai[i + k * N];
            Ar[i + k * N] = (ar * pr + ai * pi) * den;
            Ai[i + k * N] = (ai * pr - ar * pi) * den;
        }
        Grp<G>::sync();
        for (int j = k + 1 + wp; j < N; j += Grp<G>::NW) {
            const double ur = Ar[k + j * N], ui = Ai[k + j * N];
            for (int i = k + 1 + wl; i < N; i += 32) {
                const double lr = Ar[i + k * N], li = Ai[i + k * N];
                Ar[i + j * N] -= lr * ur - li * ui;
                Ai[i + j * N] -= lr * ui + li * ur;
            }
        }
        Grp<G>::sync();
    }
    return 0;
}

// ------------------------------------------------------------------------------------- LU without row moves (N <= 64)
// Rows never move: lane l of EVERY warp tracks rows l and l + 32 (rowk = elimination step at which the row was the
// pivot row, -1 before), warp w updates columns j = w (mod NW).  One barrier per elimination step.  After the
// factorisation row i with rowk = m holds its multipliers in columns j < m and U_{m,j} in columns j >= m;
// perm[k] = pivot row of step k, rd[k] = 1 / U_kk.  Multipliers of column k are written back one step late (by the
// warp that owns the column) so that no warp can still be reading the column.
struct Lu2Aux {
    int *perm, *rowk;   // [N] each
    double *rdr, *rdi;  // [N]; rdi unused for the real matrix
};
__device__ __forceinline__ Lu2Aux shp(const Lu2Aux &g)
{
    Lu2Aux x;
    x.perm = shp(g.perm); x.rowk = shp(g.rowk); x.rdr = shp(g.rdr); x.rdi = g.rdi ? shp(g.rdi) : nullptr;
    return x;
}

// exact arg-max over a warp of (key >= 0 or -1 for inactive, row index); lowest lane wins exact ties
__device__ __forceinline__ int warp_argmax_row(double v, int row)
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
    return __shfl_sync(0xffffffffu, row, __ffs(cand) - 1);
}

// exact arg-max of two independent (key, row) sets over a warp in one instruction stream: the two reductions overlap
// instead of running one after the other; exact ties (rare) take the one-set routine
__device__ __forceinline__ void warp_argmax_row2(double va, int ra, double vc, int rc, int &pa, int &pc)
{
    const bool aa = va >= 0.0, ac = vc >= 0.0;
    const unsigned ha = aa ? (unsigned)__double2hiint(va) : 0u, hc = ac ? (unsigned)__double2hiint(vc) : 0u;
    const unsigned ma = __reduce_max_sync(0xffffffffu, ha), mc = __reduce_max_sync(0xffffffffu, hc);
    const unsigned ca = __ballot_sync(0xffffffffu, aa && ha == ma), cc = __ballot_sync(0xffffffffu, ac && hc == mc);
    if (__popc(ca) == 1 && __popc(cc) == 1) {
        pa = __shfl_sync(0xffffffffu, ra, __ffs(ca) - 1);
        pc = __shfl_sync(0xffffffffu, rc, __ffs(cc) - 1);
    } else {
        pa = warp_argmax_row(va, ra);
        pc = warp_argmax_row(vc, rc);
    }
}

// Both factorisations of a Radau step in ONE pass, TWO elimination steps per sweep over the trailing matrix.
// Column-major with leading dimension LD = N + 1 (row N is a dummy row that absorbs the updates of lanes whose second
// row does not exist, so the trailing update needs no branches; rows that were pivot rows already carry a zero
// multiplier).  Lane l of EVERY warp tracks rows l and l + 32 (pivot search, reciprocals and multipliers are computed
// redundantly per warp: no exchange), warp w updates the columns j = w (mod NW).
// The trailing update is bound by shared-memory bandwidth (a load and a store per fused multiply-add), so steps k and
// k + 1 share one sweep: after the pivot of step k is known every warp updates column k + 1 for its own rows in
// registers, finds the pivot of step k + 1 there, and then each entry of the columns j >= k + 2 is loaded once, takes
//     x <- fma(-m, v', fma(-l, u, x)),   v' = fma(-t, u, v)
// (u, v = entries of the two pivot rows in column j, l, m = the row's multipliers of the two steps, t = multiplier of
// step k of pivot row k + 1) and is stored once: the operations and their order are exactly those of two rank-one
// steps, at 30 instead of 54 shared-memory wavefronts per column and with one barrier for two steps.
// Columns k and k + 1 (multipliers, and U_{k+1,k+1}) are written back one sweep late by the warps that own them, so
// that no warp can still be reading them.  perm[k] = pivot row of step k, rd[k] = 1 / U_kk.  Returns k + 1 if either
// matrix has no usable pivot at step k.
template <int G>
__device__ __noinline__ int lu2_pair(int N, int LD, double *A, const Lu2Aux &xag, double *Ar, double *Ai, const Lu2Aux &xcg)
{
    const Lu2Aux xa = shp(xag), xc = shp(xcg);
    A = shp(A); Ar = shp(Ar); Ai = shp(Ai);
    const int lane = Grp<G>::lane(), wl = Grp<G>::wlane(), wp = Grp<G>::warp();
    constexpr int NW = Grp<G>::NW;
    const int i0 = wl, i1 = wl + 32;
    const int r0 = i0 < N ? i0 : N, r1 = i1 < N ? i1 : N;             // storage rows (N = dummy)
    int ka0 = (i0 < N) ? -1 : 1 << 30, ka1 = (i1 < N) ? -1 : 1 << 30; // rowk of my two rows in the real matrix
    int kc0 = ka0, kc1 = ka1;                                         // ... in the complex matrix
    // multipliers of the first step of a sweep (column k), values for column k + 1 (multiplier or U_{k+1,k+1})
    double l0 = 0.0, l1 = 0.0, l0r = 0.0, l0i = 0.0, l1r = 0.0, l1i = 0.0;
    double w0 = 0.0, w1 = 0.0, w0r = 0.0, w0i = 0.0, w1r = 0.0, w1i = 0.0;
    auto open_after = [](int kx, int k) { return kx < 0 || (kx > k && kx < (1 << 30)); };   // row not yet a pivot row after step k
    auto write_back = [&](int k) {       // columns k, k + 1 of the sweep that started at step k
        const bool e0 = open_after(ka0, k), e1 = open_after(ka1, k), f0 = open_after(kc0, k), f1 = open_after(kc1, k);
        if (wp == k % NW) {
            if (e0) A[i0 + k * LD] = l0;
            if (e1) A[i1 + k * LD] = l1;
            if (f0) { Ar[i0 + k * LD] = l0r; Ai[i0 + k * LD] = l0i; }
            if (f1) { Ar[i1 + k * LD] = l1r; Ai[i1 + k * LD] = l1i; }
        }
        if (k + 1 < N && wp == (k + 1) % NW) {
            if (e0) A[i0 + (k + 1) * LD] = w0;
            if (e1) A[i1 + (k + 1) * LD] = w1;
            if (f0) { Ar[i0 + (k + 1) * LD] = w0r; Ai[i0 + (k + 1) * LD] = w0i; }
            if (f1) { Ar[i1 + (k + 1) * LD] = w1r; Ai[i1 + (k + 1) * LD] = w1i; }
        }
    };
    for (int k = 0; k < N; k += 2) {
        // ---- step k: pivot search in column k, reciprocals, multipliers
        const double a0 = (ka0 < 0) ? A[i0 + k * LD] : 0.0, a1 = (ka1 < 0) ? A[i1 + k * LD] : 0.0;
        const double a0r = (kc0 < 0) ? Ar[i0 + k * LD] : 0.0, a0i = (kc0 < 0) ? Ai[i0 + k * LD] : 0.0;
        const double a1r = (kc1 < 0) ? Ar[i1 + k * LD] : 0.0, a1i = (kc1 < 0) ? Ai[i1 + k * LD] : 0.0;
        const double va0 = (ka0 < 0) ? fabs(a0) : -1.0, va1 = (ka1 < 0) ? fabs(a1) : -1.0;
        const double vc0 = (kc0 < 0) ? fabs(a0r) + fabs(a0i) : -1.0, vc1 = (kc1 < 0) ? fabs(a1r) + fabs(a1i) : -1.0;
        int pa, pc;
        warp_argmax_row2(va1 > va0 ? va1 : va0, va1 > va0 ? i1 : i0, vc1 > vc0 ? vc1 : vc0, vc1 > vc0 ? i1 : i0, pa, pc);
        const double pv = (pa >= 0) ? A[pa + k * LD] : 0.0;
        const double pr = (pc >= 0) ? Ar[pc + k * LD] : 0.0, pi = (pc >= 0) ? Ai[pc + k * LD] : 0.0;
        const double den = rcp_nr(pr * pr + pi * pi);
        const double rp = rcp_nr(pv);                                 // both reciprocals before the test: they overlap
        if (pa < 0 || !isfinite(pv) || pc < 0 || !isfinite(den)) return k + 1;
        const double qr = pr * den, qi = -pi * den;                   // 1 / complex pivot
        if (i0 == pa) ka0 = k;
        if (i1 == pa) ka1 = k;
        if (i0 == pc) kc0 = k;
        if (i1 == pc) kc1 = k;
        if (lane == 0) {
            xa.perm[k] = pa; xa.rdr[k] = rp; xa.rowk[pa] = k;
            xc.perm[k] = pc; xc.rdr[k] = qr; xc.rdi[k] = qi; xc.rowk[pc] = k;
        }
        // the previous sweep's columns can be written now: every warp has passed the barrier behind its last read
        // (the values are consumed before l, w are overwritten below)
        if (k > 0) write_back(k - 2);
        l0 = (ka0 < 0) ? a0 * rp : 0.0;
        l1 = (ka1 < 0) ? a1 * rp : 0.0;
        l0r = (kc0 < 0) ? a0r * qr - a0i * qi : 0.0; l0i = (kc0 < 0) ? a0r * qi + a0i * qr : 0.0;
        l1r = (kc1 < 0) ? a1r * qr - a1i * qi : 0.0; l1i = (kc1 < 0) ? a1r * qi + a1i * qr : 0.0;
        if (k + 1 < N) {
            // ---- step k + 1: column k + 1 after step k for my rows (registers only), pivot search, multipliers
            const int kk = k + 1;
            const double uk = A[pa + kk * LD], ukr = Ar[pc + kk * LD], uki = Ai[pc + kk * LD];
            const double y0 = (ka0 < 0) ? fma(-l0, uk, A[i0 + kk * LD]) : 0.0, y1 = (ka1 < 0) ? fma(-l1, uk, A[i1 + kk * LD]) : 0.0;
            double y0r = 0.0, y0i = 0.0, y1r = 0.0, y1i = 0.0;
            if (kc0 < 0) {
                const double xr = Ar[i0 + kk * LD], xi = Ai[i0 + kk * LD];
                y0r = fma(-l0r, ukr, fma(l0i, uki, xr)); y0i = fma(-l0r, uki, fma(-l0i, ukr, xi));
            }
            if (kc1 < 0) {
                const double xr = Ar[i1 + kk * LD], xi = Ai[i1 + kk * LD];
                y1r = fma(-l1r, ukr, fma(l1i, uki, xr)); y1i = fma(-l1r, uki, fma(-l1i, ukr, xi));
            }
            const double ya0 = (ka0 < 0) ? fabs(y0) : -1.0, ya1 = (ka1 < 0) ? fabs(y1) : -1.0;
            const double yc0 = (kc0 < 0) ? fabs(y0r) + fabs(y0i) : -1.0, yc1 = (kc1 < 0) ? fabs(y1r) + fabs(y1i) : -1.0;
            int pa2, pc2;
            warp_argmax_row2(ya1 > ya0 ? ya1 : ya0, ya1 > ya0 ? i1 : i0, yc1 > yc0 ? yc1 : yc0, yc1 > yc0 ? i1 : i0, pa2, pc2);
            const int sa = pa2 < 0 ? 0 : pa2, sc = pc2 < 0 ? 0 : pc2;
            // pivot values and the step-k multipliers of the two new pivot rows sit in the lanes that hold those rows
            const double pv2 = __shfl_sync(0xffffffffu, (sa & 32) ? y1 : y0, sa & 31);
            const double tl = __shfl_sync(0xffffffffu, (sa & 32) ? l1 : l0, sa & 31);
            const double pr2 = __shfl_sync(0xffffffffu, (sc & 32) ? y1r : y0r, sc & 31);
            const double pi2 = __shfl_sync(0xffffffffu, (sc & 32) ? y1i : y0i, sc & 31);
            const double tlr = __shfl_sync(0xffffffffu, (sc & 32) ? l1r : l0r, sc & 31);
            const double tli = __shfl_sync(0xffffffffu, (sc & 32) ? l1i : l0i, sc & 31);
            const double den2 = rcp_nr(pr2 * pr2 + pi2 * pi2);
            const double rp2 = rcp_nr(pv2);
            if (pa2 < 0 || !isfinite(pv2) || pc2 < 0 || !isfinite(den2)) return kk + 1;
            const double qr2 = pr2 * den2, qi2 = -pi2 * den2;
            if (i0 == pa2) ka0 = kk;
            if (i1 == pa2) ka1 = kk;
            if (i0 == pc2) kc0 = kk;
            if (i1 == pc2) kc1 = kk;
            if (lane == 0) {
                xa.perm[kk] = pa2; xa.rdr[kk] = rp2; xa.rowk[pa2] = kk;
                xc.perm[kk] = pc2; xc.rdr[kk] = qr2; xc.rdi[kk] = qi2; xc.rowk[pc2] = kk;
            }
            const double m0 = (ka0 < 0) ? y0 * rp2 : 0.0, m1 = (ka1 < 0) ? y1 * rp2 : 0.0;
            const double m0r = (kc0 < 0) ? y0r * qr2 - y0i * qi2 : 0.0, m0i = (kc0 < 0) ? y0r * qi2 + y0i * qr2 : 0.0;
            const double m1r = (kc1 < 0) ? y1r * qr2 - y1i * qi2 : 0.0, m1i = (kc1 < 0) ? y1r * qi2 + y1i * qr2 : 0.0;
            // column k + 1 as it will be stored: U_{k+1,k+1} in the new pivot row, multipliers below
            w0 = (ka0 == kk) ? y0 : m0; w1 = (ka1 == kk) ? y1 : m1;
            w0r = (kc0 == kk) ? y0r : m0r; w0i = (kc0 == kk) ? y0i : m0i;
            w1r = (kc1 == kk) ? y1r : m1r; w1i = (kc1 == kk) ? y1i : m1i;
            // ---- both steps on the columns j >= k + 2 of this warp
            const int j0 = k + 2 + ((wp - (k + 2)) % NW + NW) % NW;
            double *c = A + j0 * LD, *cr = Ar + j0 * LD, *ci = Ai + j0 * LD;
#pragma unroll 1
            for (int j = j0; j < N; j += NW, c += NW * LD, cr += NW * LD, ci += NW * LD) {
                const double u = c[pa], v = c[pa2], x0 = c[r0], x1 = c[r1];
                const double ur = cr[pc], ui = ci[pc], vr = cr[pc2], vi = ci[pc2];
                const double x0r = cr[r0], x0i = ci[r0], x1r = cr[r1], x1i = ci[r1];
                const double v2 = fma(-tl, u, v);
                const double v2r = fma(-tlr, ur, fma(tli, ui, vr)), v2i = fma(-tlr, ui, fma(-tli, ur, vi));
                c[r0] = fma(-m0, v2, fma(-l0, u, x0));
                c[r1] = fma(-m1, v2, fma(-l1, u, x1));
                const double t0r = fma(-l0r, ur, fma(l0i, ui, x0r)), t0i = fma(-l0r, ui, fma(-l0i, ur, x0i));
                const double t1r = fma(-l1r, ur, fma(l1i, ui, x1r)), t1i = fma(-l1r, ui, fma(-l1i, ur, x1i));
                cr[r0] = fma(-m0r, v2r, fma(m0i, v2i, t0r));
                ci[r0] = fma(-m0r, v2i, fma(-m0i, v2r, t0i));
                cr[r1] = fma(-m1r, v2r, fma(m1i, v2i, t1r));
                ci[r1] = fma(-m1r, v2i, fma(-m1i, v2r, t1i));
            }
        }
        Grp<G>::sync();
    }
    write_back((N - 1) & ~1);
    Grp<G>::sync();
    // Epilogue: rows into pivot order (storage row k <- pivot row of step k) and every row of U scaled by 1 / U_kk, so
    // that a solve is two sweeps whose only chain is shuffle -> fused multiply-add: no pivot look-ups, no selects and
    // no reciprocal on the chain (solve3_*).  Column by column inside the warp that owns the column: all loads, then
    // all stores.
    {
        const bool g0 = i0 < N, g1 = i1 < N;
        const int pa0 = g0 ? xa.perm[i0] : N, pa1 = g1 ? xa.perm[i1] : N;
        const int pc0 = g0 ? xc.perm[i0] : N, pc1 = g1 ? xc.perm[i1] : N;
        const double ra0 = g0 ? xa.rdr[i0] : 0.0, ra1 = g1 ? xa.rdr[i1] : 0.0;
        const double qr0 = g0 ? xc.rdr[i0] : 0.0, qi0 = g0 ? xc.rdi[i0] : 0.0;
        const double qr1 = g1 ? xc.rdr[i1] : 0.0, qi1 = g1 ? xc.rdi[i1] : 0.0;
#pragma unroll 1
        for (int j = wp; j < N; j += NW) {
            double *c = A + j * LD, *cr = Ar + j * LD, *ci = Ai + j * LD;
            double v0 = c[pa0], v1 = c[pa1];
            double z0r = cr[pc0], z0i = ci[pc0], z1r = cr[pc1], z1i = ci[pc1];
            if (j > i0) { v0 *= ra0; const double t = z0r * qr0 - z0i * qi0; z0i = z0r * qi0 + z0i * qr0; z0r = t; }
            if (j > i1) { v1 *= ra1; const double t = z1r * qr1 - z1i * qi1; z1i = z1r * qi1 + z1i * qr1; z1r = t; }
            __syncwarp();
            if (g0) { c[i0] = v0; cr[i0] = z0r; ci[i0] = z0i; }
            if (g1) { c[i1] = v1; cr[i1] = z1r; ci[i1] = z1i; }
        }
    }
    return 0;
}

// ---- warp-specialised form of lu2_pair for a CTA of four warps: warp 0 factors the real matrix alone, warps 1-3 the
// complex one (four times the arithmetic, columns j = w (mod 3)).  In lu2_pair every warp repeats BOTH pivot chains
// (~240 instructions per elimination step, more than the trailing update); here a warp runs the chain of one matrix
// only, the two factorisations never wait for each other (the complex warps meet at a named barrier, the real warp only
// synchronises with itself), and the shared-memory traffic of the trailing updates splits about evenly (real: all
// columns x 10 wavefronts per sweep, complex: a third of the columns x 20 per warp).  Same two-steps-per-sweep
// arithmetic, pivots, result layout and return value as lu2_pair.
__device__ __forceinline__ int lu2_real_warp(int N, int LD, double *A, const Lu2Aux &xa, int wl)
{
    const int i0 = wl, i1 = wl + 32;
    const bool g0 = i0 < N, g1 = i1 < N;
    const int r0 = g0 ? i0 : N, r1 = g1 ? i1 : N;                     // storage rows (N = dummy)
    int ka0 = g0 ? -1 : 1 << 30, ka1 = g1 ? -1 : 1 << 30;
    for (int k = 0; k < N; k += 2) {
        const double a0 = (ka0 < 0) ? A[i0 + k * LD] : 0.0, a1 = (ka1 < 0) ? A[i1 + k * LD] : 0.0;
        const double va0 = (ka0 < 0) ? fabs(a0) : -1.0, va1 = (ka1 < 0) ? fabs(a1) : -1.0;
        const int pa = warp_argmax_row(va1 > va0 ? va1 : va0, va1 > va0 ? i1 : i0);
        const double pv = (pa >= 0) ? A[pa + k * LD] : 0.0;
        const double rp = rcp_nr(pv);
        if (pa < 0 || !isfinite(pv)) return k + 1;
        if (i0 == pa) ka0 = k;
        if (i1 == pa) ka1 = k;
        if (wl == 0) { xa.perm[k] = pa; xa.rdr[k] = rp; xa.rowk[pa] = k; }
        const double l0 = (ka0 < 0) ? a0 * rp : 0.0, l1 = (ka1 < 0) ? a1 * rp : 0.0;
        // a lane only ever reads its own entries of a pivot column and the pivot entry, which its owner leaves alone:
        // the multipliers can be stored at once
        if (ka0 < 0) A[i0 + k * LD] = l0;
        if (ka1 < 0) A[i1 + k * LD] = l1;
        if (k + 1 < N) {
            const int kk = k + 1;
            const double uk = A[pa + kk * LD];
            const double y0 = (ka0 < 0) ? fma(-l0, uk, A[i0 + kk * LD]) : 0.0, y1 = (ka1 < 0) ? fma(-l1, uk, A[i1 + kk * LD]) : 0.0;
            const double ya0 = (ka0 < 0) ? fabs(y0) : -1.0, ya1 = (ka1 < 0) ? fabs(y1) : -1.0;
            const int pa2 = warp_argmax_row(ya1 > ya0 ? ya1 : ya0, ya1 > ya0 ? i1 : i0);
            const int sa = pa2 < 0 ? 0 : pa2;
            const double pv2 = __shfl_sync(0xffffffffu, (sa & 32) ? y1 : y0, sa & 31);
            const double tl = __shfl_sync(0xffffffffu, (sa & 32) ? l1 : l0, sa & 31);
            const double rp2 = rcp_nr(pv2);
            if (pa2 < 0 || !isfinite(pv2)) return kk + 1;
            if (i0 == pa2) ka0 = kk;
            if (i1 == pa2) ka1 = kk;
            if (wl == 0) { xa.perm[kk] = pa2; xa.rdr[kk] = rp2; xa.rowk[pa2] = kk; }
            const double m0 = (ka0 < 0) ? y0 * rp2 : 0.0, m1 = (ka1 < 0) ? y1 * rp2 : 0.0;
            if (ka0 < 0) A[i0 + kk * LD] = m0; else if (ka0 == kk) A[i0 + kk * LD] = y0;
            if (ka1 < 0) A[i1 + kk * LD] = m1; else if (ka1 == kk) A[i1 + kk * LD] = y1;
            // four columns per trip (one warp, nothing else to hide the shared-memory round trip): all loads, then all
            // stores; a trip that runs past the last column repeats it (same values stored twice)
            double *c = A + (k + 2) * LD;
#pragma unroll 1
            for (int j = k + 2; j < N; j += 4, c += 4 * LD) {
                double *cB = c + (j + 1 < N ? LD : 0), *cC = c + (j + 2 < N ? 2 * LD : 0), *cD = c + (j + 3 < N ? 3 * LD : 0);
                const double uA = c[pa], vA = c[pa2], xA0 = c[r0], xA1 = c[r1];
                const double uB = cB[pa], vB = cB[pa2], xB0 = cB[r0], xB1 = cB[r1];
                const double uC = cC[pa], vC = cC[pa2], xC0 = cC[r0], xC1 = cC[r1];
                const double uD = cD[pa], vD = cD[pa2], xD0 = cD[r0], xD1 = cD[r1];
                const double wA = fma(-tl, uA, vA), wB = fma(-tl, uB, vB), wC = fma(-tl, uC, vC), wD = fma(-tl, uD, vD);
                __syncwarp();                                         // every lane has read the pivot rows
                c[r0] = fma(-m0, wA, fma(-l0, uA, xA0));
                c[r1] = fma(-m1, wA, fma(-l1, uA, xA1));
                cB[r0] = fma(-m0, wB, fma(-l0, uB, xB0));
                cB[r1] = fma(-m1, wB, fma(-l1, uB, xB1));
                cC[r0] = fma(-m0, wC, fma(-l0, uC, xC0));
                cC[r1] = fma(-m1, wC, fma(-l1, uC, xC1));
                cD[r0] = fma(-m0, wD, fma(-l0, uD, xD0));
                cD[r1] = fma(-m1, wD, fma(-l1, uD, xD1));
            }
        }
        __syncwarp();
    }
    // rows into pivot order, U scaled by 1 / U_kk (see lu2_pair)
    const int p0 = g0 ? xa.perm[i0] : N, p1 = g1 ? xa.perm[i1] : N;
    const double rd0 = g0 ? xa.rdr[i0] : 0.0, rd1 = g1 ? xa.rdr[i1] : 0.0;
#pragma unroll 2
    for (int j = 0; j < N; j++) {
        double *c = A + j * LD;
        double v0 = c[p0], v1 = c[p1];
        if (j > i0) v0 *= rd0;
        if (j > i1) v1 *= rd1;
        __syncwarp();
        if (g0) c[i0] = v0;
        if (g1) c[i1] = v1;
    }
    return 0;
}

// NWc warps (wq = 0 .. NWc-1) on the complex matrix; they meet at named barrier 1
__device__ __forceinline__ int lu2_complex_warps(int N, int LD, double *Ar, double *Ai, const Lu2Aux &xc, int wl, int wq, int NWc)
{
    auto bar = [&]() { asm volatile("bar.sync 1, %0;" ::"r"(NWc * 32) : "memory"); };
    const int i0 = wl, i1 = wl + 32;
    const bool g0 = i0 < N, g1 = i1 < N;
    const int r0 = g0 ? i0 : N, r1 = g1 ? i1 : N;
    int kc0 = g0 ? -1 : 1 << 30, kc1 = g1 ? -1 : 1 << 30;
    double l0r = 0.0, l0i = 0.0, l1r = 0.0, l1i = 0.0, w0r = 0.0, w0i = 0.0, w1r = 0.0, w1i = 0.0;
    auto open_after = [](int kx, int k) { return kx < 0 || (kx > k && kx < (1 << 30)); };
    auto write_back = [&](int k) {       // columns k, k + 1 of the sweep that started at step k (owner warps, one sweep late)
        const bool f0 = open_after(kc0, k), f1 = open_after(kc1, k);
        if (wq == k % NWc) {
            if (f0) { Ar[i0 + k * LD] = l0r; Ai[i0 + k * LD] = l0i; }
            if (f1) { Ar[i1 + k * LD] = l1r; Ai[i1 + k * LD] = l1i; }
        }
        if (k + 1 < N && wq == (k + 1) % NWc) {
            if (f0) { Ar[i0 + (k + 1) * LD] = w0r; Ai[i0 + (k + 1) * LD] = w0i; }
            if (f1) { Ar[i1 + (k + 1) * LD] = w1r; Ai[i1 + (k + 1) * LD] = w1i; }
        }
    };
    for (int k = 0; k < N; k += 2) {
        const double a0r = (kc0 < 0) ? Ar[i0 + k * LD] : 0.0, a0i = (kc0 < 0) ? Ai[i0 + k * LD] : 0.0;
        const double a1r = (kc1 < 0) ? Ar[i1 + k * LD] : 0.0, a1i = (kc1 < 0) ? Ai[i1 + k * LD] : 0.0;
        const double vc0 = (kc0 < 0) ? fabs(a0r) + fabs(a0i) : -1.0, vc1 = (kc1 < 0) ? fabs(a1r) + fabs(a1i) : -1.0;
        const int pc = warp_argmax_row(vc1 > vc0 ? vc1 : vc0, vc1 > vc0 ? i1 : i0);
        const double pr = (pc >= 0) ? Ar[pc + k * LD] : 0.0, pi = (pc >= 0) ? Ai[pc + k * LD] : 0.0;
        const double den = rcp_nr(pr * pr + pi * pi);
        if (pc < 0 || !isfinite(den)) return k + 1;
        const double qr = pr * den, qi = -pi * den;                   // 1 / pivot
        if (i0 == pc) kc0 = k;
        if (i1 == pc) kc1 = k;
        if (wq == 0 && wl == 0) { xc.perm[k] = pc; xc.rdr[k] = qr; xc.rdi[k] = qi; xc.rowk[pc] = k; }
        if (k > 0) write_back(k - 2);
        l0r = (kc0 < 0) ? a0r * qr - a0i * qi : 0.0; l0i = (kc0 < 0) ? a0r * qi + a0i * qr : 0.0;
        l1r = (kc1 < 0) ? a1r * qr - a1i * qi : 0.0; l1i = (kc1 < 0) ? a1r * qi + a1i * qr : 0.0;
        if (k + 1 < N) {
            const int kk = k + 1;
            const double ukr = Ar[pc + kk * LD], uki = Ai[pc + kk * LD];
            double y0r = 0.0, y0i = 0.0, y1r = 0.0, y1i = 0.0;
            if (kc0 < 0) {
                const double xr = Ar[i0 + kk * LD], xi = Ai[i0 + kk * LD];
                y0r = fma(-l0r, ukr, fma(l0i, uki, xr)); y0i = fma(-l0r, uki, fma(-l0i, ukr, xi));
            }
            if (kc1 < 0) {
                const double xr = Ar[i1 + kk * LD], xi = Ai[i1 + kk * LD];
                y1r = fma(-l1r, ukr, fma(l1i, uki, xr)); y1i = fma(-l1r, uki, fma(-l1i, ukr, xi));
            }
            const double yc0 = (kc0 < 0) ? fabs(y0r) + fabs(y0i) : -1.0, yc1 = (kc1 < 0) ? fabs(y1r) + fabs(y1i) : -1.0;
            const int pc2 = warp_argmax_row(yc1 > yc0 ? yc1 : yc0, yc1 > yc0 ? i1 : i0);
            const int sc = pc2 < 0 ? 0 : pc2;
            const double pr2 = __shfl_sync(0xffffffffu, (sc & 32) ? y1r : y0r, sc & 31);
            const double pi2 = __shfl_sync(0xffffffffu, (sc & 32) ? y1i : y0i, sc & 31);
            const double tlr = __shfl_sync(0xffffffffu, (sc & 32) ? l1r : l0r, sc & 31);
            const double tli = __shfl_sync(0xffffffffu, (sc & 32) ? l1i : l0i, sc & 31);
            const double den2 = rcp_nr(pr2 * pr2 + pi2 * pi2);
            if (pc2 < 0 || !isfinite(den2)) return kk + 1;
            const double qr2 = pr2 * den2, qi2 = -pi2 * den2;
            if (i0 == pc2) kc0 = kk;
            if (i1 == pc2) kc1 = kk;
            if (wq == 0 && wl == 0) { xc.perm[kk] = pc2; xc.rdr[kk] = qr2; xc.rdi[kk] = qi2; xc.rowk[pc2] = kk; }
            const double m0r = (kc0 < 0) ? y0r * qr2 - y0i * qi2 : 0.0, m0i = (kc0 < 0) ? y0r * qi2 + y0i * qr2 : 0.0;
            const double m1r = (kc1 < 0) ? y1r * qr2 - y1i * qi2 : 0.0, m1i = (kc1 < 0) ? y1r * qi2 + y1i * qr2 : 0.0;
            w0r = (kc0 == kk) ? y0r : m0r; w0i = (kc0 == kk) ? y0i : m0i;
            w1r = (kc1 == kk) ? y1r : m1r; w1i = (kc1 == kk) ? y1i : m1i;
            const int j0 = k + 2 + ((wq - (k + 2)) % NWc + NWc) % NWc;
            double *cr = Ar + j0 * LD, *ci = Ai + j0 * LD;
#pragma unroll 1
            for (int j = j0; j < N; j += NWc, cr += NWc * LD, ci += NWc * LD) {
                const double ur = cr[pc], ui = ci[pc], vr = cr[pc2], vi = ci[pc2];
                const double x0r = cr[r0], x0i = ci[r0], x1r = cr[r1], x1i = ci[r1];
                const double v2r = fma(-tlr, ur, fma(tli, ui, vr)), v2i = fma(-tlr, ui, fma(-tli, ur, vi));
                const double t0r = fma(-l0r, ur, fma(l0i, ui, x0r)), t0i = fma(-l0r, ui, fma(-l0i, ur, x0i));
                const double t1r = fma(-l1r, ur, fma(l1i, ui, x1r)), t1i = fma(-l1r, ui, fma(-l1i, ur, x1i));
                __syncwarp();                                         // every lane has read the two pivot rows
                cr[r0] = fma(-m0r, v2r, fma(m0i, v2i, t0r));
                ci[r0] = fma(-m0r, v2i, fma(-m0i, v2r, t0i));
                cr[r1] = fma(-m1r, v2r, fma(m1i, v2i, t1r));
                ci[r1] = fma(-m1r, v2i, fma(-m1i, v2r, t1i));
            }
        }
        bar();
    }
    write_back((N - 1) & ~1);
    bar();
    const int p0 = g0 ? xc.perm[i0] : N, p1 = g1 ? xc.perm[i1] : N;
    const double q0r = g0 ? xc.rdr[i0] : 0.0, q0i = g0 ? xc.rdi[i0] : 0.0, q1r = g1 ? xc.rdr[i1] : 0.0, q1i = g1 ? xc.rdi[i1] : 0.0;
#pragma unroll 1
    for (int j = wq; j < N; j += NWc) {
        double *cr = Ar + j * LD, *ci = Ai + j * LD;
        double z0r = cr[p0], z0i = ci[p0], z1r = cr[p1], z1i = ci[p1];
        if (j > i0) { const double t = z0r * q0r - z0i * q0i; z0i = z0r * q0i + z0i * q0r; z0r = t; }
        if (j > i1) { const double t = z1r * q1r - z1i * q1i; z1i = z1r * q1i + z1i * q1r; z1r = t; }
        __syncwarp();
        if (g0) { cr[i0] = z0r; ci[i0] = z0i; }
        if (g1) { cr[i1] = z1r; ci[i1] = z1i; }
    }
    return 0;
}

// one CTA of 128 threads; includes the barrier behind the factorisation
__device__ __noinline__ int lu2_split(int N, int LD, double *A, const Lu2Aux &xag, double *Ar, double *Ai, const Lu2Aux &xcg)
{
    const Lu2Aux xa = shp(xag), xc = shp(xcg);
    A = shp(A); Ar = shp(Ar); Ai = shp(Ai);
    const int wl = threadIdx.x & 31, wp = threadIdx.x >> 5;
    int ier;
    if (wp == 0) ier = lu2_real_warp(N, LD, A, xa, wl);
    else ier = lu2_complex_warps(N, LD, Ar, Ai, xc, wl, wp - 1, 3);
    return __syncthreads_or(ier);
}

// Solves with the factors as lu2_pair leaves them (rows in pivot order, unit-diagonal scaled U): b (shared, length N,
// original row order) is overwritten by x.  Lane l holds components l and l + 32; step k broadcasts component k
// and every later (earlier) row subtracts its multiple: the chain per step is one shuffle and one fused multiply-add
// (two for the complex system).  Entries outside the triangle are masked to zero when they are loaded, off the chain.
__device__ __forceinline__ void solve3_real_warp(int N, int LD, const double *A, const Lu2Aux &x, double *b, int wl)
{
    const int i0 = wl, i1 = wl + 32;
    const bool g0 = i0 < N, g1 = i1 < N;
    const int r0 = g0 ? i0 : N, r1 = g1 ? i1 : N;       // storage rows (N = dummy row of the lu2 layout)
    double b0 = g0 ? b[x.perm[i0]] : 0.0, b1 = g1 ? b[x.perm[i1]] : 0.0;
    const double rd0 = g0 ? x.rdr[i0] : 0.0, rd1 = g1 ? x.rdr[i1] : 0.0;
    const int K1 = N - 1 < 32 ? N - 1 : 32;
    // the matrix entries of the NEXT step are requested before the broadcast of this one (unconditional loads: the
    // other triangle and the dummy row are valid memory), so that only shuffle -> fused multiply-add is on the chain
    const double *a0 = A + r0, *a1 = A + r1;
    double n0 = *a0, n1 = *a1;
    int k = 0;
#pragma unroll 2
    for (; k < K1; k++) {
        const double l0 = (i0 > k) ? n0 : 0.0, l1 = g1 ? n1 : 0.0;
        a0 += LD; a1 += LD;
        n0 = *a0; n1 = *a1;
        const double bk = __shfl_sync(0xffffffffu, b0, k);
        b0 = fma(-l0, bk, b0);
        b1 = fma(-l1, bk, b1);
    }
#pragma unroll 2
    for (; k < N - 1; k++) {
        const double l1 = (g1 && i1 > k) ? n1 : 0.0;
        a1 += LD;
        n1 = *a1;
        const double bk = __shfl_sync(0xffffffffu, b1, k - 32);
        b1 = fma(-l1, bk, b1);
    }
    b0 *= rd0; b1 *= rd1;
    k = N - 1;
    a0 = A + r0 + k * LD; a1 = A + r1 + k * LD;
    n0 = *a0; n1 = *a1;
#pragma unroll 2
    for (; k >= 32; k--) {
        const double u0 = n0, u1 = (i1 < k) ? n1 : 0.0;
        a0 -= LD; a1 -= LD;
        n0 = *a0; n1 = *a1;
        const double xk = __shfl_sync(0xffffffffu, b1, k - 32);
        b0 = fma(-u0, xk, b0);
        b1 = fma(-u1, xk, b1);
    }
#pragma unroll 2
    for (; k >= 1; k--) {
        const double u0 = (i0 < k) ? n0 : 0.0;
        a0 -= LD;
        n0 = *a0;
        const double xk = __shfl_sync(0xffffffffu, b0, k);
        b0 = fma(-u0, xk, b0);
    }
    __syncwarp();
    if (g0) b[i0] = b0;
    if (g1) b[i1] = b1;
    __syncwarp();
}
__device__ __forceinline__ void solve3_complex_warp(int N, int LD, const double *Ar, const double *Ai, const Lu2Aux &x, double *br,
                                                    double *bi, int wl)
{
    const int i0 = wl, i1 = wl + 32;
    const bool g0 = i0 < N, g1 = i1 < N;
    const int r0 = g0 ? i0 : N, r1 = g1 ? i1 : N;
    const int p0 = g0 ? x.perm[i0] : 0, p1 = g1 ? x.perm[i1] : 0;
    double b0r = g0 ? br[p0] : 0.0, b0i = g0 ? bi[p0] : 0.0, b1r = g1 ? br[p1] : 0.0, b1i = g1 ? bi[p1] : 0.0;
    const double q0r = g0 ? x.rdr[i0] : 0.0, q0i = g0 ? x.rdi[i0] : 0.0, q1r = g1 ? x.rdr[i1] : 0.0, q1i = g1 ? x.rdi[i1] : 0.0;
    const int K1 = N - 1 < 32 ? N - 1 : 32;
    int o0 = r0, o1 = r1;
    double n0r = Ar[o0], n0i = Ai[o0], n1r = Ar[o1], n1i = Ai[o1];      // entries of the next step, requested early
    int k = 0;
#pragma unroll 2
    for (; k < K1; k++) {
        const bool m0 = i0 > k;
        const double l0r = m0 ? n0r : 0.0, l0i = m0 ? n0i : 0.0, l1r = g1 ? n1r : 0.0, l1i = g1 ? n1i : 0.0;
        o0 += LD; o1 += LD;
        n0r = Ar[o0]; n0i = Ai[o0]; n1r = Ar[o1]; n1i = Ai[o1];
        const double xr = __shfl_sync(0xffffffffu, b0r, k), xi = __shfl_sync(0xffffffffu, b0i, k);
        b0r = fma(-l0r, xr, fma(l0i, xi, b0r));
        b0i = fma(-l0r, xi, fma(-l0i, xr, b0i));
        b1r = fma(-l1r, xr, fma(l1i, xi, b1r));
        b1i = fma(-l1r, xi, fma(-l1i, xr, b1i));
    }
#pragma unroll 2
    for (; k < N - 1; k++) {
        const bool m1 = g1 && i1 > k;
        const double l1r = m1 ? n1r : 0.0, l1i = m1 ? n1i : 0.0;
        o1 += LD;
        n1r = Ar[o1]; n1i = Ai[o1];
        const double xr = __shfl_sync(0xffffffffu, b1r, k - 32), xi = __shfl_sync(0xffffffffu, b1i, k - 32);
        b1r = fma(-l1r, xr, fma(l1i, xi, b1r));
        b1i = fma(-l1r, xi, fma(-l1i, xr, b1i));
    }
    { const double t = b0r * q0r - b0i * q0i; b0i = b0r * q0i + b0i * q0r; b0r = t; }
    { const double t = b1r * q1r - b1i * q1i; b1i = b1r * q1i + b1i * q1r; b1r = t; }
    k = N - 1;
    o0 = r0 + k * LD; o1 = r1 + k * LD;
    n0r = Ar[o0]; n0i = Ai[o0]; n1r = Ar[o1]; n1i = Ai[o1];
#pragma unroll 2
    for (; k >= 32; k--) {
        const bool m1 = i1 < k;
        const double u0r = n0r, u0i = n0i, u1r = m1 ? n1r : 0.0, u1i = m1 ? n1i : 0.0;
        o0 -= LD; o1 -= LD;
        n0r = Ar[o0]; n0i = Ai[o0]; n1r = Ar[o1]; n1i = Ai[o1];
        const double xr = __shfl_sync(0xffffffffu, b1r, k - 32), xi = __shfl_sync(0xffffffffu, b1i, k - 32);
        b0r = fma(-u0r, xr, fma(u0i, xi, b0r));
        b0i = fma(-u0r, xi, fma(-u0i, xr, b0i));
        b1r = fma(-u1r, xr, fma(u1i, xi, b1r));
        b1i = fma(-u1r, xi, fma(-u1i, xr, b1i));
    }
#pragma unroll 2
    for (; k >= 1; k--) {
        const bool m0 = i0 < k;
        const double u0r = m0 ? n0r : 0.0, u0i = m0 ? n0i : 0.0;
        o0 -= LD;
        n0r = Ar[o0]; n0i = Ai[o0];
        const double xr = __shfl_sync(0xffffffffu, b0r, k), xi = __shfl_sync(0xffffffffu, b0i, k);
        b0r = fma(-u0r, xr, fma(u0i, xi, b0r));
        b0i = fma(-u0r, xi, fma(-u0i, xr, b0i));
    }
    __syncwarp();
    if (g0) { br[i0] = b0r; bi[i0] = b0i; }
    if (g1) { br[i1] = b1r; bi[i1] = b1i; }
    __syncwarp();
}
template <int G>
__device__ __noinline__ void solve2_pair(int N, int LD, const double *E1, const Lu2Aux &x1g, double *z1, const double *E2r,
                                         const double *E2i, const Lu2Aux &x2g, double *z2, double *z3)
{
    const Lu2Aux x1 = shp(x1g), x2 = shp(x2g);     // everything below is dynamic shared memory
    E1 = shp(E1); E2r = shp(E2r); E2i = shp(E2i); z1 = shp(z1); z2 = shp(z2); z3 = shp(z3);
    if (G == 32) {
        solve3_real_warp(N, LD, E1, x1, z1, Grp<G>::wlane());
        solve3_complex_warp(N, LD, E2r, E2i, x2, z2, z3, Grp<G>::wlane());
    } else {
        if (Grp<G>::warp() == 0) solve3_real_warp(N, LD, E1, x1, z1, Grp<G>::wlane());
        else if (Grp<G>::warp() == 1) solve3_complex_warp(N, LD, E2r, E2i, x2, z2, z3, Grp<G>::wlane());
    }
    Grp<G>::sync();
}
template <int G>
__device__ __noinline__ void solve2_real(int N, int LD, const double *E1, const Lu2Aux &x1g, double *b)
{
    const Lu2Aux x1 = shp(x1g);
    E1 = shp(E1); b = shp(b);
    if (Grp<G>::warp() == 0) solve3_real_warp(N, LD, E1, x1, b, Grp<G>::wlane());
    Grp<G>::sync();
}

// Solves by ONE warp (lanes wl = 0..31) on shared vectors; P b first, then L, then U (column sweeps).
__device__ __forceinline__ void solve_real_warp(int N, const double *A, const int *ip, double *b, int wl)
{
    if (wl == 0)
        for (int k = 0; k < N; k++) {
            const int p = ip[k];
            const double tmp = b[p];
            b[p] = b[k];
            b[k] = tmp;
        }
    __syncwarp();
    for (int k = 0; k < N - 1; k++) {
        const double bk = b[k];
        for (int i = k + 1 + wl; i < N; i += 32) b[i] -= A[i + k * N] * bk;
        __syncwarp();
    }
    for (int k = N - 1; k >= 0; k--) {
        const double bk = b[k] / A[k + k * N];
        __syncwarp();
        if (wl == 0) b[k] = bk;
        for (int i = wl; i < k; i += 32) b[i] -= A[i + k * N] * bk;
        __syncwarp();
    }
}
__device__ __forceinline__ void solve_complex_warp(int N, const double *Ar, const double *Ai, const int *ip, double *br,
                                                   double *bi, int wl)
{
    if (wl == 0)
        for (int k = 0; k < N; k++) {
            const int p = ip[k];
            double tmp = br[p];
            br[p] = br[k];
            br[k] = tmp;
            tmp = bi[p];
            bi[p] = bi[k];
            bi[k] = tmp;
        }
    __syncwarp();
    for (int k = 0; k < N - 1; k++) {
        const double xr = br[k], xi = bi[k];
        for (int i = k + 1 + wl; i < N; i += 32) {
            const double lr = Ar[i + k * N], li = Ai[i + k * N];
            br[i] -= lr * xr - li * xi;
            bi[i] -= lr * xi + li * xr;
        }
        __syncwarp();
    }
    for (int k = N - 1; k >= 0; k--) {
        const double pr = Ar[k + k * N], pi = Ai[k + k * N];
        const double den = 1.0 / (pr * pr + pi * pi);
        const double vr = br[k], vi = bi[k];
        const double xr = (vr * pr + vi * pi) * den, xi = (vi * pr - vr * pi) * den;
        __syncwarp();
        if (wl == 0) { br[k] = xr; bi[k] = xi; }
        for (int i = wl; i < k; i += 32) {
            const double ur = Ar[i + k * N], ui = Ai[i + k * N];
            br[i] -= ur * xr - ui * xi;
            bi[i] -= ur * xi + ui * xr;
        }
        __syncwarp();
    }
}

// One real and one complex solve for the group: a single warp does both when G == 32, warps 0 and 1
// work side by side when the group is a CTA.
template <int G>
__device__ __noinline__ void solve_pair(int N, const double *E1, const int *ip1, double *z1, const double *E2r,
                                           const double *E2i, const int *ip2, double *z2, double *z3)
{
    if (G == 32) {
        solve_real_warp(N, E1, ip1, z1, Grp<G>::wlane());
        solve_complex_warp(N, E2r, E2i, ip2, z2, z3, Grp<G>::wlane());
    } else {
        if (Grp<G>::warp() == 0) solve_real_warp(N, E1, ip1, z1, Grp<G>::wlane());
        else if (Grp<G>::warp() == 1) solve_complex_warp(N, E2r, E2i, ip2, z2, z3, Grp<G>::wlane());
    }
    Grp<G>::sync();
}
template <int G>
__device__ __noinline__ void solve_real(int N, const double *E1, const int *ip1, double *b)
{
    if (Grp<G>::warp() == 0) solve_real_warp(N, E1, ip1, b, Grp<G>::wlane());
    Grp<G>::sync();
}

}  // namespace chem

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
// the first version of this kernel was bound by instruction-cache misses (profiles/r1_history.md).
#pragma once
#include "chem_radau.cuh"

namespace chem {

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
__device__ __noinline__ double exp_ni(double a) { return exp_f(a); }
__device__ __noinline__ double log_ni(double a) { return log_f(a); }
// a^b for normal a > 0 (step-size controller only): exp(b ln a) from the compact routines above, ~|b ln a| ulp;
// the library pow() is a 270-instruction routine that this instruction-fetch-bound kernel would stream in twice per step
__device__ __forceinline__ double pow_ni(double a, double b) { return exp_ni(b * log_ni(a)); }

// per-warp scratch layout (doubles), three stage slots each: C[3][32] (C[s][31] = 1 for unused factor slots),
// E[3][64] exp-job results, q[3][32] rates of progress, X[48] stage parameters and phase-2 jobs; then matrices
constexpr int kWsC = 0, kWsE = 96, kWsQ = kWsE + 3 * kJobs, kWsX = kWsQ + 96, kWsMat = kWsX + 48;

// Mixture front end shared by the source term and the Jacobian: returns T, fills C[], E[] (exp jobs).
struct WarpMix {
    double T, lnT, invT, rho, inv_rho, Wbar, Ck, invWk;
    const double *spc, *jt;
    bool lo;
};
__device__ __forceinline__ WarpMix warp_front(const double *tab, double *ws, double tmid, double P, double invP, double yc,
                                              int lane, int N)
{
    WarpMix m;
    double *C = ws + kWsC, *E = ws + kWsE;
    m.T = __shfl_sync(0xffffffffu, yc, 0);
    double Yk = __shfl_down_sync(0xffffffffu, yc, 1);     // species lane k holds Y_k = component k+1
    if (lane >= N - 1) Yk = 0.0;
    m.lo = (m.T <= tmid);
    const double *spt = tab + (m.lo ? kOffSpLo : kOffSpHi);
    m.spc = spt + (lane < N ? lane : 0) * kJobW;
    m.invWk = m.spc[7];
    double sY = Yk, sYW = Yk * m.invWk;
    warp_sum2(sY, sYW);
    const double YN = 1.0 - sY;                            // closure: last species
    if (lane == N - 1) Yk = YN;
    const double sW = sYW + YN * spt[(N - 1) * kJobW + 7]; // 1 / Wbar
    m.Wbar = rcp_f(sW);
    m.invT = rcp_f(m.T);
    m.rho = P * m.Wbar * m.invT * (1.0 / kRerg);
    m.inv_rho = kRerg * m.T * sW * invP;
    m.lnT = m.T > 0.0 ? log_ni(m.T) : __longlong_as_double(0x7ff8000000000000LL);
    m.Ck = m.rho * Yk * m.invWk;
    if (lane < N) C[lane] = m.Ck;
    m.jt = tab + (m.lo ? kOffJobLo : kOffJobHi);
#pragma unroll 1
    for (int r = 0; r < 2; r++)
        E[32 * r + lane] = exp_ni(job_arg(m.jt + (32 * r + lane) * kJobW, m.T, m.lnT, m.invT));
    __syncwarp();
    return m;
}

struct D3 { double a, b, c; };

// Source term at THREE states at once (the three Radau stage points of one Newton iteration):
// component `lane` of stage s is y.a / y.b / y.c (lane 0: T, lanes 1..N-1: Y_1..Y_{N-1}); returns component
// `lane` of the three f.  DESIGN.md R1-R5; same mathematics as rhs<G>() in chem_device.cuh.
// Batching the stages lets one instruction stream serve 3 x 64 exp jobs, lets single lanes take the serial
// transcendentals (ln T, reciprocals, the Troe broadening factor of every (reaction, stage) pair) in
// parallel, and shares every table read.  tab = staged table blob (shared), ws = this warp's scratch (shared).
template <int NS>
__device__ __forceinline__ D3 warp_rhs_body(const double *tab, double *ws, double tmid, double P, double invP, D3 y)
{
    const int lane = threadIdx.x & 31;
    const int *hdr = reinterpret_cast<const int *>(tab);
    const int N = hdr[0];
    const int4 d0 = reinterpret_cast<const int4 *>(tab + kOffDesc)[lane];       // factors, troe ordinal, type, jobs
    const int4 d1 = reinterpret_cast<const int4 *>(tab + kOffDesc)[32 + lane];   // eff_lo, eff_hi, inc_lo, inc_hi
    double *C = ws + kWsC, *E = ws + kWsE, *q = ws + kWsQ, *X = ws + kWsX;
    const int row = lane < N ? lane : 0;
    double T[NS], Yk[NS], sY[NS], sYW[NS];
    const double yin[3] = {y.a, y.b, y.c};
#pragma unroll
    for (int s = 0; s < NS; s++) {
        T[s] = __shfl_sync(0xffffffffu, yin[s], 0);
        Yk[s] = __shfl_down_sync(0xffffffffu, yin[s], 1);
    }
    const double invWk = tab[kOffSpLo + row * kJobW + 7], invWN = tab[kOffSpLo + (N - 1) * kJobW + 7];
#pragma unroll
    for (int s = 0; s < NS; s++) {
        if (lane >= N - 1) Yk[s] = 0.0;
        sY[s] = Yk[s];
        sYW[s] = Yk[s] * invWk;
    }
#pragma unroll 1
    for (int o = 16; o > 0; o >>= 1)      // rolled on purpose: code size matters more than the loop overhead here
#pragma unroll
        for (int s = 0; s < NS; s++) {
            sY[s] += __shfl_xor_sync(0xffffffffu, sY[s], o);
            sYW[s] += __shfl_xor_sync(0xffffffffu, sYW[s], o);
        }
    double sW[NS];
#pragma unroll
    for (int s = 0; s < NS; s++) {
        const double YN = 1.0 - sY[s];                      // closure: last species
        if (lane == N - 1) Yk[s] = YN;
        sW[s] = sYW[s] + YN * invWN;                        // 1 / Wbar
    }
    // serial transcendentals, one lane each: lanes 0-2 take T_s (ln, 1/x), lanes 3-5 take 1/Wbar_s (1/x)
    const int sl3 = lane % NS;
    double Tsel = T[0], Wsel = sW[0];
#pragma unroll
    for (int s = 1; s < NS; s++)
        if (sl3 == s) { Tsel = T[s]; Wsel = sW[s]; }
    const double lnsel = Tsel > 0.0 ? log_f(Tsel) : __longlong_as_double(0x7ff8000000000000LL);   // a stage T <= 0 is a failed step (R11), as with libm's log
    const double rsel = rcp_f((lane >= NS && lane < 2 * NS) ? Wsel : Tsel);
    double invT[NS], rho[NS], inv_rho[NS], Ck[NS];
#pragma unroll
    for (int s = 0; s < NS; s++) {
        invT[s] = __shfl_sync(0xffffffffu, rsel, s);
        const double Wbar = __shfl_sync(0xffffffffu, rsel, NS + s);
        const double lnT = __shfl_sync(0xffffffffu, lnsel, s);
        rho[s] = P * Wbar * invT[s] * (1.0 / kRerg);
        inv_rho[s] = kRerg * T[s] * sW[s] * invP;
        Ck[s] = rho[s] * Yk[s] * invWk;
        if (lane < N) C[32 * s + lane] = Ck[s];
        if (lane == 0) { X[4 * s] = T[s]; X[4 * s + 1] = lnT; X[4 * s + 2] = invT[s]; }
    }
    __syncwarp();
    // exp jobs: 3 stages x 2 rounds per lane, one rolled loop
#pragma unroll 1
    for (int it = 0; it < 2 * NS; it++) {
        const int s = it >> 1, r = it & 1;
        const double Ts = X[4 * s], lnT = X[4 * s + 1], iT = X[4 * s + 2];
        const double *c = tab + (Ts <= tmid ? kOffJobLo : kOffJobHi) + (32 * r + lane) * kJobW;
        E[kJobs * s + 32 * r + lane] = exp_f(job_arg(c, Ts, lnT, iT));
    }
    __syncwarp();
    // rates of progress of reaction `lane` at the three stages; factors: species indices with multiplicity, 31 = unity
    const int type = d0.z;
    double rnet[NS], cm[NS];
#pragma unroll
    for (int s = 0; s < NS; s++) { rnet[s] = 0.0; cm[s] = 1.0; }
    if (type >= 0) {
#pragma unroll
        for (int s = 0; s < NS; s++) {
            const double *Cs = C + 32 * s, *Es = E + kJobs * s;
            const double Rf = Es[lane] * (Cs[d0.x & 31] * Cs[(d0.x >> 5) & 31] * Cs[(d0.x >> 10) & 31]);
            const double Rr = Es[32 + lane] * (Cs[(d0.x >> 15) & 31] * Cs[(d0.x >> 20) & 31] * Cs[(d0.x >> 25) & 31]);
            rnet[s] = Rf - Rr;
        }
        if (type != 0) {
            const double *eff_dv = tab + hdr[4];
            const int *eff_sp = reinterpret_cast<const int *>(tab + hdr[5]);
#pragma unroll
            for (int s = 0; s < NS; s++) cm[s] = P * invT[s] * (1.0 / kRerg);
#pragma unroll 1
            for (int p = d1.x; p < d1.y; p++) {
                const double dv = eff_dv[p];
                const int sp = eff_sp[p];
                #pragma unroll
                for (int s = 0; s < NS; s++) cm[s] += dv * C[32 * s + sp];
            }
            if (type >= 2) {
                // hand (Fcent, Pr) of every (reaction, stage) pair to the phase-2 lanes; Lindemann: Fcent = 1
                const int slot = 12 + 2 * NS * d0.y;
#pragma unroll
                for (int s = 0; s < NS; s++) {
                    const double *Es = E + kJobs * s;
                    const int ts = (d0.w >> 8) & 255;
                    X[slot + 2 * s] = type == 3 ? Es[ts] + Es[ts + 1] + Es[ts + 2] : 1.0;
                    X[slot + 2 * s + 1] = Es[d0.w & 255] * cm[s];
                }
            }
        }
    }
    __syncwarp();
    // phase 2: lane pair (2p, 2p+1) serves falloff pair p = (ordinal, stage): c = Pr/(1+Pr) F  (R5)
    {
        const int nfo = hdr[7];                                   // number of falloff reactions
        const bool live = lane < 2 * NS * nfo;
        const double v = live ? X[12 + lane] : 1.0;
        const double lg = log_f(v) * kInvLn10;                      // even lane: log10 Fcent, odd lane: log10 Pr
        const double lPr = __shfl_down_sync(0xffffffffu, lg, 1);
        const double Pr = __shfl_down_sync(0xffffffffu, v, 1);
        const double At = lPr - 0.4 - 0.67 * lg;
        const double x = At * rcp_f(0.75 - 1.27 * lg - 0.14 * At);
        const double F = exp_f(kLn10 * lg * rcp_f(1.0 + x * x));
        const double c = Pr * rcp_f(1.0 + Pr) * F;
        __syncwarp();
        if (live && !(lane & 1)) X[12 + lane] = c;
    }
    __syncwarp();
    if (type >= 2) {
        const int slot = 12 + 2 * NS * d0.y;
        #pragma unroll
        for (int s = 0; s < NS; s++) cm[s] = X[slot + 2 * s];
    }
#pragma unroll
    for (int s = 0; s < NS; s++) q[32 * s + lane] = type >= 0 ? cm[s] * rnet[s] : 0.0;
    __syncwarp();
    // species production rates (three stages per pass over the incidence list), temperature equation
    const int2 *inc = reinterpret_cast<const int2 *>(tab + hdr[3]);      // (reaction, net stoichiometric coefficient)
    double w[NS];
#pragma unroll
    for (int s = 0; s < NS; s++) w[s] = 0.0;
#pragma unroll 1
    for (int p = d1.z; p < d1.w; p++) {
        const int2 e = inc[p];
        const double nu = (double)e.y;
        #pragma unroll
        for (int s = 0; s < NS; s++) w[s] += nu * q[32 * s + e.x];
    }
    double hw[NS], ccp[NS];
#pragma unroll
    for (int s = 0; s < NS; s++) {
        const double *spc = tab + (T[s] <= tmid ? kOffSpLo : kOffSpHi) + row * kJobW;
        const double Ts = T[s];
        const double cpR = spc[0] + Ts * (spc[1] + Ts * (spc[2] + Ts * (spc[3] + Ts * spc[4])));
        const double hRT = spc[0] + Ts * (spc[1] * 0.5 + Ts * (spc[2] * (1.0 / 3.0) + Ts * (spc[3] * 0.25 + Ts * (spc[4] * 0.2)))) + spc[5] * invT[s];
        hw[s] = lane < N ? hRT * w[s] : 0.0;
        ccp[s] = lane < N ? Ck[s] * cpR : 0.0;
    }
#pragma unroll 1
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int s = 0; s < NS; s++) {
            hw[s] += __shfl_xor_sync(0xffffffffu, hw[s], o);
            ccp[s] += __shfl_xor_sync(0xffffffffu, ccp[s], o);
        }
    const double Wk = tab[kOffSpLo + row * kJobW + 6];
    double csel = ccp[0];
#pragma unroll
    for (int s = 1; s < NS; s++)
        if (sl3 == s) csel = ccp[s];
    const double rc = rcp_f(csel);
    double f[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int s = 0; s < NS; s++) {
        const double Ydot = Wk * w[s] * inv_rho[s];               // W_k wdot_k / rho in species lane k
        f[s] = __shfl_up_sync(0xffffffffu, Ydot, 1);               // component k+1
        const double rccp = __shfl_sync(0xffffffffu, rc, s);
        if (lane == 0) f[s] = -T[s] * hw[s] * rccp;
    }
    __syncwarp();
    D3 out;
    out.a = f[0]; out.b = f[1]; out.c = f[2];
    return out;
}

// out-of-line instances: the Newton iterations evaluate three stage points at once, everything else one state
// (a one-state call runs and fetches about a third of the instructions; the kernel is bound by instruction fetch)
__device__ __noinline__ D3 warp_rhs3(const double *tab, double *ws, double tmid, double P, double invP, D3 y)
{
    return warp_rhs_body<3>(tab, ws, tmid, P, invP, y);
}
__device__ __noinline__ double warp_rhs1(const double *tab, double *ws, double tmid, double P, double invP, double y)
{
    return warp_rhs_body<1>(tab, ws, tmid, P, invP, D3{y, y, y}).a;
}

// Analytical Jacobian (R6) for the warp path: Jm[i*N + j] = d f_i / d y_j in shared memory.
// Temperature derivatives of all rate constants come from the exp-job rows (d/dT exp(p(T)) = p'(T) exp(p(T))).
// scr: 8*32 doubles (dq[6][32], dqdT[32], tb[32]); vec: 3*16 doubles (wdot, hRT, cpR per species).
__device__ __noinline__ void warp_jacobian(const double *tab, double *ws, double tmid, double P, double invP, double yc,
                                           double *Jm, double *scr, double *vec)
{
    const int lane = threadIdx.x & 31;
    const int *hdr = reinterpret_cast<const int *>(tab);
    const int N = hdr[0];
    const int4 *desc = reinterpret_cast<const int4 *>(tab + kOffDesc);
    const int4 d0 = desc[lane], d1 = desc[32 + lane];
    double *C = ws + kWsC, *E = ws + kWsE, *q = ws + kWsQ;
    double *dq = scr, *dqdT = scr + 192, *tb = scr + 224;
    const double *eff_dv = tab + hdr[4];
    const int *eff_sp = reinterpret_cast<const int *>(tab + hdr[5]);
    const WarpMix m = warp_front(tab, ws, tmid, P, invP, yc, lane, N);
    const double T = m.T, invT = m.invT;
    const double Ctot = P * invT * (1.0 / kRerg);
    {
        double qi = 0.0, dT = 0.0, tbi = 0.0, d[6] = {0, 0, 0, 0, 0, 0};
        const int type = d0.z;
        if (type >= 0) {
            const double c0 = C[d0.x & 31], c1 = C[(d0.x >> 5) & 31], c2 = C[(d0.x >> 10) & 31];
            const double c3 = C[(d0.x >> 15) & 31], c4 = C[(d0.x >> 20) & 31], c5 = C[(d0.x >> 25) & 31];
            const double kf = E[lane], kr = E[32 + lane];
            const double Rf = kf * (c0 * c1 * c2), Rr = kr * (c3 * c4 * c5), rnet = Rf - Rr;
            const double dlnkf = job_darg(m.jt + lane * kJobW, T, invT), dlnkr = job_darg(m.jt + (32 + lane) * kJobW, T, invT);
            double c = 1.0, dc_dT = 0.0, dc_dM = 0.0;
            if (type != 0) {
                double M = Ctot;
#pragma unroll 1
                for (int p = d1.x; p < d1.y; p++) M += eff_dv[p] * C[eff_sp[p]];
                c = M;
                dc_dM = 1.0;
                if (type >= 2) {
                    const int ks = d0.w & 255;
                    const double k0k = E[ks], Pr = k0k * M, dlnPr = job_darg(m.jt + ks * kJobW, T, invT);
                    double F = 1.0, dF_dT = 0.0, dF_dPr = 0.0;
                    if (type == 3) {
                        const int ts = (d0.w >> 8) & 255;
                        const double e3 = E[ts], e1 = E[ts + 1], e2 = E[ts + 2];
                        const double Fc = e3 + e1 + e2;
                        const double dFc = e3 * job_darg(m.jt + ts * kJobW, T, invT) + e1 * job_darg(m.jt + (ts + 1) * kJobW, T, invT) +
                                           e2 * job_darg(m.jt + (ts + 2) * kJobW, T, invT);
                        const double L = log_ni(Fc) * kInvLn10, dL = dFc * rcp_f(Fc) * kInvLn10;
                        const double At = log_ni(Pr) * kInvLn10 - 0.4 - 0.67 * L;
                        const double Bt = 0.75 - 1.27 * L - 0.14 * At, rB = rcp_f(Bt);
                        const double x = At * rB, rden = rcp_f(1.0 + x * x);
                        F = exp_ni(kLn10 * L * rden);
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
            qi = c * rnet;
            dT = dc_dT * rnet + c * (Rf * dlnkf - Rr * dlnkr);
            tbi = dc_dM * rnet;
            const double ckf = c * kf, ckr = -c * kr;
            d[0] = ckf * c1 * c2; d[1] = ckf * c0 * c2; d[2] = ckf * c0 * c1;
            d[3] = ckr * c4 * c5; d[4] = ckr * c3 * c5; d[5] = ckr * c3 * c4;
        }
        q[lane] = qi; dqdT[lane] = dT; tb[lane] = (type > 0) ? tbi : 0.0;
#pragma unroll
        for (int sl = 0; sl < 6; sl++) dq[sl * 32 + lane] = d[sl];
    }
    __syncwarp();
    // rows: species lane k -> Dw[k][j] = d wdot_k / d y_j, stored in Jm row k
    const double *spt = tab + (m.lo ? kOffSpLo : kOffSpHi);
    const double *spc = m.spc;
    const double invWN = spt[(N - 1) * kJobW + 7];
    const double cpR = spc[0] + T * (spc[1] + T * (spc[2] + T * (spc[3] + T * spc[4])));
    const double dcpR = spc[1] + T * (2.0 * spc[2] + T * (3.0 * spc[3] + T * (4.0 * spc[4])));
    const double hRT = spc[0] + T * (spc[1] * 0.5 + T * (spc[2] * (1.0 / 3.0) + T * (spc[3] * 0.25 + T * (spc[4] * 0.2)))) + spc[5] * invT;
    double hw = 0.0, ccp = 0.0, cpw = 0.0, cdcp = 0.0;
    if (lane < N) {
        const int2 *inc = reinterpret_cast<const int2 *>(tab + hdr[3]);
        double *row = Jm + lane * N;
#pragma unroll 1
        for (int l = 0; l < N; l++) row[l] = 0.0;
        double wd = 0.0, dwT = 0.0, u = 0.0;
#pragma unroll 1
        for (int p = d1.z; p < d1.w; p++) {
            const int i = inc[p].x;
            const double nu = (double)inc[p].y;
            const int4 e0 = desc[i], e1 = desc[32 + i];
            wd += nu * q[i];
            dwT += nu * dqdT[i];
#pragma unroll
            for (int sl = 0; sl < 6; sl++) {
                const int f = (e0.x >> (5 * sl)) & 31;
                if (f != 31) row[f] += nu * dq[sl * 32 + i];
            }
            const double v = nu * tb[i];
            u += v;
#pragma unroll 1
            for (int pe = e1.x; pe < e1.y; pe++) row[eff_sp[pe]] += v * eff_dv[pe];
        }
        double GC = 0.0;
#pragma unroll 1
        for (int l = 0; l < N; l++) GC += row[l] * C[l];
        const double GN = row[N - 1] * invWN;
#pragma unroll 1
        for (int j = N - 1; j >= 1; j--) {
            const double iw = spt[(j - 1) * kJobW + 7];
            row[j] = -m.Wbar * (iw - invWN) * GC + m.rho * (row[j - 1] * iw - GN);
        }
        row[0] = dwT - (GC + u * Ctot) * invT;
        vec[lane] = wd; vec[16 + lane] = hRT; vec[32 + lane] = cpR;
        hw = hRT * wd; ccp = m.Ck * cpR; cpw = cpR * wd; cdcp = m.Ck * dcpR;
    }
    warp_sum2(hw, ccp);
    warp_sum2(cpw, cdcp);
    __syncwarp();
    const double rccp = rcp_f(ccp);
    const double Tdot = -T * hw * rccp;
    // columns: assemble the rows of J in place (row k+1 <- species k, descending; row 0 <- temperature)
    if (lane < N) {
        const int j = lane;
        double S = 0.0;
#pragma unroll 1
        for (int k = 0; k < N; k++) S += vec[16 + k] * Jm[k * N + j];
        double dlnrho, drcp;
        if (j == 0) {
            dlnrho = -invT;
            drcp = -ccp * invT + cdcp;
        } else {
            const double iw = spt[(j - 1) * kJobW + 7];
            dlnrho = -m.Wbar * (iw - invWN);
            drcp = dlnrho * ccp + m.rho * (vec[32 + j - 1] * iw - vec[32 + N - 1] * invWN);
        }
#pragma unroll 1
        for (int k = N - 2; k >= 0; k--) {
            const double Wr = spt[k * kJobW + 6] * m.inv_rho;
            Jm[(k + 1) * N + j] = Wr * (Jm[k * N + j] - vec[k] * dlnrho);
        }
        Jm[j] = -(T * S + (j == 0 ? cpw : 0.0)) * rccp - Tdot * drcp * rccp;
    }
    __syncwarp();
}

// ---------------------------------------------------------------------------- linear algebra with rows owned by lanes
// Separate arg-max in each half-warp with FULL-mask collectives only (partial-mask reductions take a slow
// WARPSYNC path): returns the row 0..15 of the maximum of key v (>= 0, or -1 for inactive lanes) within the
// caller's half h, or -1 if that maximum is not > 0.  Highest word first, low word on ties, lowest row wins exact ties.
__device__ __forceinline__ int half_argmax(double v, int h)
{
    const bool act = v >= 0.0;
    const unsigned hi = act ? (unsigned)__double2hiint(v) : 0u;
    const unsigned m0 = __reduce_max_sync(0xffffffffu, h ? 0u : hi), m1 = __reduce_max_sync(0xffffffffu, h ? hi : 0u);
    const unsigned m = h ? m1 : m0;
    unsigned cand = (__ballot_sync(0xffffffffu, act && hi == m) >> (16 * h)) & 0xffffu;
    if (__any_sync(0xffffffffu, __popc(cand) != 1)) {
        const unsigned lo = (act && hi == m) ? (unsigned)__double2loint(v) : 0u;
        const unsigned l0 = __reduce_max_sync(0xffffffffu, h ? 0u : lo), l1 = __reduce_max_sync(0xffffffffu, h ? lo : 0u);
        const unsigned m2 = h ? l1 : l0;
        cand = (__ballot_sync(0xffffffffu, act && hi == m && lo == m2) >> (16 * h)) & 0xffffu;
        if (m == 0u && m2 == 0u) cand = 0u;
    }
    return cand ? __ffs(cand) - 1 : -1;
}

// Gauss-Jordan inversion of BOTH Radau matrices in one instruction stream: half-warp 0 handles the real matrix E1
// (imaginary parts zero), half-warp 1 the complex matrix E2, both with complex arithmetic ("LU
// factorization of the Jacobian"; one real and one complex N x N system per step).  The elimination is the one of LU
// with partial pivoting on |re| + |im| (R10: same pivot sequence), continued above the diagonal, so that each
// of the ~9 solves per factorisation becomes a matrix-vector product without the 2N-long chain of dependent
// broadcasts of a triangular solve (the one place where this path departs from the oracle's
// arithmetic; the group kernels keep LU + triangular solves).  Z[h][N][LD] complex (re, im); row r of half h is owned by lane
// 16 h + r and never moves.  With p_k the pivot row of step k, the row operations G satisfy G A = D Pi (row p_k of
// the result is piv_k e_k^T), so A^-1 = Pi^T D^-1 G.  In place: column k of the storage ends as column p_k of G.
// Outputs: myk = step at which this lane's row was the pivot row, (rdr, rdi) = 1/piv of that row, src = lane owning
// the pivot row of step r (where component r of a solution is produced).  Returns 0, or k + 1 at a zero/non-finite pivot.
__device__ __noinline__ int gj_warp_pair(double2 *Z, int LD, int N, int &myk_out, int &src_out, double &rdr_out, double &rdi_out)
{
    const int lane = threadIdx.x & 31, h = lane >> 4, r = lane & 15;
    double2 *Zh = Z + h * N * LD;
    double2 *row = Zh + (r < N ? r : 0) * LD;
    int myk = -1, src = lane;
    double rdr = 0.0, rdi = 0.0;
    for (int k = 0; k < N; k++) {
        const double2 a = row[k];
        const int p = half_argmax((r < N && myk < 0) ? fabs(a.x) + fabs(a.y) : -1.0, h);
        const double2 *prow = Zh + (p < 0 ? 0 : p) * LD;
        const double2 pv = prow[k];
        const double den = rcp_f(pv.x * pv.x + pv.y * pv.y);
        if (__any_sync(0xffffffffu, p < 0 || !isfinite(den))) return k + 1;
        const double qr = pv.x * den, qi = -pv.y * den;       // 1 / pivot
        if (r == k) src = 16 * h + p;
        if (r == p) { myk = k; rdr = qr; rdi = qi; }
        if (r < N && r != p) {
            const double lr = a.x * qr - a.y * qi, li = a.x * qi + a.y * qr;
            const double2 *u = prow;
            double2 *x = row;
#pragma unroll 1
            for (int n = N; n > 0; n--, u++, x++) {
                const double2 uu = *u;
                double2 xx = *x;
                xx.x = fma(-lr, uu.x, fma(li, uu.y, xx.x));
                xx.y = fma(-lr, uu.y, fma(-li, uu.x, xx.y));
                *x = xx;
            }
            row[k] = make_double2(-lr, -li);                   // column p_k of G (the eliminated entry itself is zero)
        }
        __syncwarp();
        if (r == p) row[k] = make_double2(1.0, 0.0);           // only its owner reads this row from now on
    }
    myk_out = myk;
    src_out = src;
    rdr_out = rdr;
    rdi_out = rdi;
    return 0;
}

// Solve with both inverses at once: lane 16 h + r passes row r of the right-hand side of system h and receives
// component r of its solution.  bp: 34 complex scratch entries (b permuted to pivot order, one dump slot per half).
__device__ __noinline__ double2 solve_warp_pair(const double2 *Z, int LD, int N, double2 *bp, int myk, int src, double rdr,
                                                double rdi, double br, double bi)
{
    const int lane = threadIdx.x & 31, h = lane >> 4, r = lane & 15;
    const double2 *x = Z + h * N * LD + (r < N ? r : 0) * LD;
    double2 *bh = bp + 17 * h;
    bh[myk >= 0 ? myk : 16] = make_double2(br, bi);
    __syncwarp();
    double ar = 0.0, ai = 0.0, cr = 0.0, ci = 0.0;
    const double2 *b = bh;
#pragma unroll 1
    for (int n = N; n > 0; n--, b++, x++) {
        const double2 bb = *b, g = *x;
        ar = fma(g.x, bb.x, ar);
        cr = fma(-g.y, bb.y, cr);
        ai = fma(g.x, bb.y, ai);
        ci = fma(g.y, bb.x, ci);
    }
    ar += cr;
    ai += ci;
    const double vr = ar * rdr - ai * rdi, vi = ar * rdi + ai * rdr;      // component myk of the solution
    __syncwarp();
    return make_double2(__shfl_sync(0xffffffffu, vr, src), __shfl_sync(0xffffffffu, vi, src));
}

}  // namespace chem

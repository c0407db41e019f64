// chem_cta.cuh -- stage-batched source term for the group kernels (G = 32 or 128 threads per state), built on the
// exp-job tables of the mechanism compiler (chem.cu): the three Radau stage states of one Newton iteration are
// evaluated in one pass, every rate constant is one exp of a 7-term form in T, the Troe broadening
// factors of all (falloff reaction, stage) pairs are computed side by side by separate threads.
// Same mathematics as rhs<G>() (R1-R5).
#pragma once
#include "chem_device.cuh"

namespace chem {

// extra shared scratch of the batched source term (doubles): ys2, ys3, C3[3][64], X0[3][8], X[3][n_fo][4], q3[3][NR], red6[6 NW]
__host__ __device__ inline size_t cta_extra_doubles(int N, int NR, int n_fo, int NW)
{
    // (C3 shares the six chemistry vectors of the Jacobian routine, q3 extends its q: see carve())
    return (size_t)2 * N + (6 * N < 192 ? 192 - 6 * N : 0) + 24 + (size_t)12 * (n_fo > 0 ? n_fo : 1) + (size_t)2 * NR + 6 * NW + 2;
}

struct CtaScratch {
    double *ys2, *ys3;   // stage states 2, 3 (stage 1 is Work::ys)
    double *C3;          // [3][64], C3[s][63] = 1 (unity factor)
    double *X0;          // [3][8]: T, lnT, 1/T, rho, 1/rho, Ctot
    double *X;           // [3][n_fo][4]: Fcent, Pr, rnet, reaction index
    double *q3;          // [3][NR]
    double *red6;        // [6][NW]
};

// block all-reduce of six sums (deterministic: fixed butterfly, then warps in order)
template <int G>
__device__ __forceinline__ void sum6(double (&v)[6], double *red6)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int c = 0; c < 6; c++) v[c] += __shfl_xor_sync(0xffffffffu, v[c], o);
    if (G > 32) {
        __syncthreads();
        if (Grp<G>::wlane() == 0)
#pragma unroll
            for (int c = 0; c < 6; c++) red6[c * Grp<G>::NW + Grp<G>::warp()] = v[c];
        __syncthreads();
#pragma unroll
        for (int c = 0; c < 6; c++) {
            double a = 0.0;
#pragma unroll
            for (int wv = 0; wv < Grp<G>::NW; wv++) a += red6[c * Grp<G>::NW + wv];
            v[c] = a;
        }
    }
}

struct JobRow { double2 c01, c23, c45, c67; };
__device__ __forceinline__ JobRow job_load(const double *c)
{
    JobRow r;
    r.c01 = __ldg(reinterpret_cast<const double2 *>(c)); r.c23 = __ldg(reinterpret_cast<const double2 *>(c) + 1);
    r.c45 = __ldg(reinterpret_cast<const double2 *>(c) + 2); r.c67 = __ldg(reinterpret_cast<const double2 *>(c) + 3);
    return r;
}
__device__ __forceinline__ double job_eval(const JobRow &r, double T, double lnT, double invT)
{
    return exp_f(r.c01.x + r.c01.y * lnT + r.c23.x * invT + T * (r.c23.y + T * (r.c45.x + T * (r.c45.y + T * r.c67.x))));
}
__device__ __forceinline__ double job_val(const double *c, double T, double lnT, double invT)
{
    return job_eval(job_load(c), T, lnT, invT);
}

// Inputs: stage states ys[0..2] (shared, length N); outputs f[0..2] (shared, length N).  nstage = 1 or 3.
template <int G>
__device__ __noinline__ void cta_rhs3(const Tables &tg, const ChemScratch &cs, const CtaScratch &xg, double P, int nstage,
                                      const double *ys0, double *f0, double *f1, double *f2)
{
    const Tables &t = *shp(&tg);     // the kernel's shared copy of the descriptor
    const int N = t.n_sp, NR = t.n_rx, nfo = t.n_fo;
    const int lane = Grp<G>::lane();
    CtaScratch x;        // all of these live in dynamic shared memory: say so to the compiler (shp)
    x.ys2 = shp(xg.ys2); x.ys3 = shp(xg.ys3); x.C3 = shp(xg.C3); x.X0 = shp(xg.X0); x.X = shp(xg.X); x.q3 = shp(xg.q3);
    x.red6 = shp(xg.red6);
    ys0 = shp(ys0); f0 = shp(f0); f1 = shp(f1); f2 = shp(f2);
    const double *ys[3] = {ys0, x.ys2, x.ys3};
    double *fo[3] = {f0, f1, f2};
    // ---- mixture: closure, Wbar, rho, concentrations
    double v[6] = {0, 0, 0, 0, 0, 0};
    for (int k = lane; k < N - 1; k += G) {
        const double iw = __ldg(&t.invW[k]);
#pragma unroll
        for (int s = 0; s < 3; s++)
            if (s < nstage) { const double Yk = ys[s][k + 1]; v[2 * s] += Yk; v[2 * s + 1] += Yk * iw; }
    }
    sum6<G>(v, x.red6);
    if (lane < nstage) {
        const int s = lane;
        const double T = (s == 0 ? ys0 : (s == 1 ? x.ys2 : x.ys3))[0];
        const double vY = s == 0 ? v[0] : (s == 1 ? v[2] : v[4]), vW = s == 0 ? v[1] : (s == 1 ? v[3] : v[5]);
        const double YN = 1.0 - vY;
        const double sW = vW + YN * __ldg(&t.invW[N - 1]);
        const double invT = 1.0 / T, rho = P / (kRerg * T * sW);
        double *o = x.X0 + 8 * s;
        o[0] = T; o[2] = invT; o[3] = rho; o[4] = kRerg * T * sW / P; o[5] = P * invT * (1.0 / kRerg);
        o[1] = T > 0.0 ? log_f(T) : __longlong_as_double(0x7ff8000000000000LL);   // a stage T <= 0 is a failed step (R11), as with libm's log
        x.C3[64 * s + N - 1] = rho * YN * __ldg(&t.invW[N - 1]);
        x.C3[64 * s + 63] = 1.0;
    }
    Grp<G>::sync();
    for (int k = lane; k < N - 1; k += G) {
        const double iw = __ldg(&t.invW[k]);
#pragma unroll
        for (int s = 0; s < 3; s++)
            if (s < nstage) x.C3[64 * s + k] = x.X0[8 * s + 3] * ys[s][k + 1] * iw;
    }
    Grp<G>::sync();
    // ---- rates of progress.  Work units of equal cost (six exps) and one kind per warp, so that no warp runs two
    // branches one after the other while the rest of the group waits at the barrier:
    //   (1) one (falloff reaction, stage) pair per thread: k_f, k_r, k_0/k_inf and the three Troe terms of ONE stage
    //       (table reactions [0, n_fo) are the falloff reactions: Troe first, then Lindemann);
    //   (2) one elementary / three-body reaction per thread with ALL stages (two exps per stage), coefficient rows read
    //       once; the threads behind the last warp that got a falloff pair start first.
    const int nft = nfo * nstage;
    for (int q = lane; q < nft; q += G) {
        const int s = q / nfo, i = q - s * nfo;
        const int4 d0 = __ldg(reinterpret_cast<const int4 *>(t.rdesc) + 2 * i);       // f012, f345, type, extra job
        const int4 d1 = __ldg(reinterpret_cast<const int4 *>(t.rdesc) + 2 * i + 1);   // falloff ordinal, eff_lo, eff_hi
        const double T = x.X0[8 * s], lnT = x.X0[8 * s + 1], invT = x.X0[8 * s + 2];
        const double *jt = (T <= t.tmid0) ? t.job_lo : t.job_hi;
        const double *C = x.C3 + 64 * s;
        const JobRow rf = job_load(jt + (size_t)i * 8), rr = job_load(jt + (size_t)(NR + i) * 8), r0 = job_load(jt + (size_t)d0.w * 8);
        const double kf = job_eval(rf, T, lnT, invT), kr = job_eval(rr, T, lnT, invT);
        const double Rf = kf * (C[d0.x & 255] * C[(d0.x >> 8) & 255] * C[(d0.x >> 16) & 255]);
        const double Rr = kr * (C[d0.y & 255] * C[(d0.y >> 8) & 255] * C[(d0.y >> 16) & 255]);
        double M = x.X0[8 * s + 5];
#pragma unroll 4
        for (int p = d1.y; p < d1.z; p++) M += __ldg(&t.eff_dv[p]) * C[__ldg(&t.eff_sp[p])];
        const double Pr = job_eval(r0, T, lnT, invT) * M;
        double Fc = 1.0;
        if (d0.z == 3)
            Fc = job_val(jt + (size_t)(d0.w + 1) * 8, T, lnT, invT) + job_val(jt + (size_t)(d0.w + 2) * 8, T, lnT, invT) +
                 job_val(jt + (size_t)(d0.w + 3) * 8, T, lnT, invT);
        double *o = x.X + (size_t)(s * nfo + d1.x) * 4;
        o[0] = Fc; o[1] = Pr; o[2] = Rf - Rr; o[3] = (double)i;
    }
    const int used = nft % G, head = (used + 31) & ~31;                // threads of the last falloff trip, in whole warps
    const int vt = lane >= head ? lane - head : lane + (G - head);     // virtual thread index of part (2)
    for (int i = nfo + vt; i < NR; i += G) {
        const int4 d0 = __ldg(reinterpret_cast<const int4 *>(t.rdesc) + 2 * i);
        const int4 d1 = __ldg(reinterpret_cast<const int4 *>(t.rdesc) + 2 * i + 1);
        // the coefficient rows of k_f and k_r are read once for all stages when the stages share a NASA range (the rule;
        // job tables live in L2: 49 KB per range for the GRI shape)
        const double *jt0 = (x.X0[0] <= t.tmid0) ? t.job_lo : t.job_hi;
        const JobRow rf = job_load(jt0 + (size_t)i * 8), rr = job_load(jt0 + (size_t)(NR + i) * 8);
#pragma unroll 1
        for (int s = 0; s < nstage; s++) {
            const double T = x.X0[8 * s], lnT = x.X0[8 * s + 1], invT = x.X0[8 * s + 2];
            const double *jt = (T <= t.tmid0) ? t.job_lo : t.job_hi;
            const double *C = x.C3 + 64 * s;
            double kf, kr;
            if (jt == jt0) { kf = job_eval(rf, T, lnT, invT); kr = job_eval(rr, T, lnT, invT); }
            else { kf = job_val(jt + (size_t)i * 8, T, lnT, invT); kr = job_val(jt + (size_t)(NR + i) * 8, T, lnT, invT); }
            const double Rf = kf * (C[d0.x & 255] * C[(d0.x >> 8) & 255] * C[(d0.x >> 16) & 255]);
            const double Rr = kr * (C[d0.y & 255] * C[(d0.y >> 8) & 255] * C[(d0.y >> 16) & 255]);
            double c = 1.0;
            if (d0.z != 0) {
                double M = x.X0[8 * s + 5];
#pragma unroll 4
                for (int p = d1.y; p < d1.z; p++) M += __ldg(&t.eff_dv[p]) * C[__ldg(&t.eff_sp[p])];   // unrolled: loads batched
                c = M;
            }
            x.q3[s * NR + i] = c * (Rf - Rr);
        }
    }
    Grp<G>::sync();
    // ---- falloff pairs (reaction, stage): c = Pr/(1+Pr) F, one thread each (R5)
    for (int p = lane; p < nstage * nfo; p += G) {
        const double *o = x.X + (size_t)p * 4;
        const double Fc = o[0], Pr = o[1];
        const double L = log_f(Fc) * kInvLn10;
        const double At = log_f(Pr) * kInvLn10 - 0.4 - 0.67 * L;
        const double xx = At * rcp_nr(0.75 - 1.27 * L - 0.14 * At);
        const double F = exp_f(kLn10 * L * rcp_nr(1.0 + xx * xx));
        const int s = p / nfo;
        x.q3[s * NR + (int)o[3]] = Pr * rcp_nr(1.0 + Pr) * F * o[2];
    }
    Grp<G>::sync();
    // ---- species production rates, temperature equation
    double r6[6] = {0, 0, 0, 0, 0, 0};
    auto species_tail = [&](int k, const double (&w)[3]) {
        const double Wk = __ldg(&t.W[k]);
#pragma unroll
        for (int s = 0; s < 3; s++)
            if (s < nstage) {
                const double T = x.X0[8 * s], invT = x.X0[8 * s + 2];
                const double *a = (T <= t.tmid0) ? t.nasa_lo : t.nasa_hi;
                const double a0 = __ldg(&a[k]), a1 = __ldg(&a[N + k]), a2 = __ldg(&a[2 * N + k]), a3 = __ldg(&a[3 * N + k]);
                const double a4 = __ldg(&a[4 * N + k]), a5 = __ldg(&a[5 * N + k]);
                const double cpR = a0 + T * (a1 + T * (a2 + T * (a3 + T * a4)));
                const double hRT = a0 + T * (a1 * 0.5 + T * (a2 * (1.0 / 3.0) + T * (a3 * 0.25 + T * (a4 * 0.2)))) + a5 * invT;
                r6[2 * s] += hRT * w[s];
                r6[2 * s + 1] += x.C3[64 * s + k] * cpR;
                if (k < N - 1) fo[s][k + 1] = Wk * w[s] * x.X0[8 * s + 4];
            }
    };
    if (t.gat_steps >= 0) {
        // balanced gather (schedule built by the mechanism compiler): the incidence list of a species is shared by
        // 2^g.w adjacent threads; long lists (radicals that take part in a third of the reactions) no longer hold the
        // whole group at the next barrier
        const int4 g = __ldg(t.gat + lane);
        double w[3] = {0.0, 0.0, 0.0};
#pragma unroll 4
        for (int p = g.y; p < g.z; p++) {
            const int2 e = __ldg(t.inc2 + p);
            const double nu = (double)e.y;
#pragma unroll
            for (int s = 0; s < 3; s++)
                if (s < nstage) w[s] += nu * x.q3[s * NR + e.x];
        }
        for (int o = 1; o < (1 << t.gat_steps); o <<= 1) {
#pragma unroll
            for (int s = 0; s < 3; s++) {
                const double v = __shfl_xor_sync(0xffffffffu, w[s], o);
                if (o < (1 << g.w)) w[s] += v;
            }
        }
        if (g.x >= 0 && (lane & ((1 << g.w) - 1)) == 0) species_tail(g.x, w);
    } else {
        for (int k = lane; k < N; k += G) {
            double w[3] = {0.0, 0.0, 0.0};
            for (int p = __ldg(&t.inc_ptr[k]); p < __ldg(&t.inc_ptr[k + 1]); p++) {
                const double nu = __ldg(&t.inc_nu[p]);
                const int i = __ldg(&t.inc_rx[p]);
#pragma unroll
                for (int s = 0; s < 3; s++)
                    if (s < nstage) w[s] += nu * x.q3[s * NR + i];
            }
            species_tail(k, w);
        }
    }
    sum6<G>(r6, x.red6);
    if (lane < nstage) {
        const double hw = lane == 0 ? r6[0] : (lane == 1 ? r6[2] : r6[4]), ccp = lane == 0 ? r6[1] : (lane == 1 ? r6[3] : r6[5]);
        (lane == 0 ? f0 : (lane == 1 ? f1 : f2))[0] = -x.X0[8 * lane] * hw / ccp;
    }
    Grp<G>::sync();
    (void)cs;
}

}  // namespace chem

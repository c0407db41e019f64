// chem_common.cuh -- definitions shared by every kernel family of the path (group, warp-per-state, thread-per-state):
// physical constants, the packed device tables written by the mechanism compiler, the exp-job table layout, the Radau IIA
// method constants (R7) and the parameter / result records of one integration.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

#include "chem_math.cuh"

namespace chem {

constexpr double kRerg = 8.31446261815324e7;  // erg/(mol K)
constexpr double kRcal = 1.98720425864083;    // cal/(mol K)
constexpr double kPatm = 1.01325e6;           // dyn/cm^2
constexpr int kSlots = 6;                     // 3 reactant + 3 product slots per reaction

// Packed device tables written by the mechanism compiler (chem_mech_load).
struct Tables {
    int n_sp, n_rx;
    const double *W, *invW;           // [n_sp]
    const double *nasa_lo, *nasa_hi;  // [7][n_sp], coefficient-major
    const double *tmid;               // [n_sp]
    const int *rtype;                 // [n_rx]
    const double *lnA, *b, *Ta;       // [n_rx]  ln A, b, Ea/R [K]
    const double *lnA0, *b0, *Ta0;    // [n_rx]  low-pressure limit
    const double *dnu;                // [n_rx]  sum nu'' - sum nu'
    const double *troe;               // [4][n_rx]
    const int *slot_sp, *slot_nu;     // [6][n_rx]; slots 0-2 reactants, 3-5 products; unused: sp 0, nu 0
    const int *eff_ptr, *eff_sp;      // CSR over reactions
    const double *eff_dv;             // alpha - 1
    const int *inc_ptr, *inc_rx;      // CSR over species: reactions the species takes part in
    const double *inc_nu;             // net stoichiometric coefficient nu'' - nu'
    // exp-job form of the rate constants (chem_cta.cuh); n_jobs == 0: not available for this mechanism
    const double *job_lo, *job_hi;    // [n_jobs][8]: k_f [0,n_rx), k_r [n_rx,2 n_rx), then k_0/k_inf and Troe terms
    const int *rdesc;                 // [n_rx][8]: factors 0-2 (8 bits each, 63 = unity), factors 3-5, type, extra job, falloff ordinal, eff_lo, eff_hi, 0
    int n_jobs, n_fo;
    double tmid0;
    // balanced gather schedule of cta_rhs3 (chem.cu): per thread of a group (species or -1, first entry, end, log2 of the
    // species' thread count); inc2 = (reaction, net coefficient) pairs in inc_ptr order; gat_steps = max log2, -1: none
    const int4 *gat;
    const int2 *inc2;
    int gat_steps;
    int n_solo;                       // threads t < n_solo evaluate table reaction t only (chem.cu)
    // balanced row gather of the analytical Jacobian (jacobian<128>): schedule like `gat` for gatj_T threads (0: none),
    // jinc = two int4 per incidence: (reaction, net coefficient, slot species 0-2, slot species 3-5), (eff_lo, eff_hi, has [M], 0)
    const int4 *gatj;
    const int4 *jinc;
    int gatj_T;
};

constexpr int kJobW = 9;     // doubles per job row (7 used; 8 for species rows); ODD: lane-per-row reads are bank-conflict free
constexpr int kJobs = 64;    // 2 rounds x 32 lanes
// fixed part of the staged table blob (doubles)
constexpr int kOffJobLo = 8, kOffJobHi = kOffJobLo + kJobs * kJobW, kOffSpLo = kOffJobHi + kJobs * kJobW;
constexpr int kOffSpHi = kOffSpLo + 16 * kJobW, kOffDesc = kOffSpHi + 16 * kJobW;   // desc: 2 planes x 32 lanes x int4 = 128 doubles
constexpr int kOffLists = kOffDesc + 128;

// Tables of the fast path: one blob in global memory, staged into shared memory once per CTA.
// blob[0..7] is a header of ints: {n_sp, n_rx, off_inc_nu, off_inc (int pairs), off_eff_dv, off_eff_sp, LD, n_falloff} (offsets in doubles).
struct FastTables {
    int enabled;
    int n_sp, n_rx;
    int blob_doubles;
    double tmid;             // common NASA switch temperature
    const double *blob;
};

// exponent of job row c at T and its temperature derivative
__device__ __forceinline__ double job_arg(const double *c, double T, double lnT, double invT)
{
    return c[0] + c[1] * lnT + c[2] * invT + T * (c[3] + T * (c[4] + T * (c[5] + T * c[6])));
}
__device__ __forceinline__ double job_darg(const double *c, double T, double invT)
{
    return (c[1] - c[2] * invT) * invT + c[3] + T * (2.0 * c[4] + T * (3.0 * c[5] + T * (4.0 * c[6])));
}

// Method constants (R7).  The real matrices T, T^-1 block-diagonalise A^-1 into
// gamma (real) and alpha +- i beta; values to 20 digits from Hairer & Wanner, Sec. IV.8.
namespace rk {
constexpr double SQ6 = 2.449489742783178098;
constexpr double C1 = (4.0 - SQ6) / 10.0, C2 = (4.0 + SQ6) / 10.0;
constexpr double C1M1 = C1 - 1.0, C2M1 = C2 - 1.0, C1MC2 = C1 - C2;
constexpr double DD1 = -(13.0 + 7.0 * SQ6) / 3.0, DD2 = (-13.0 + 7.0 * SQ6) / 3.0, DD3 = -1.0 / 3.0;
// 1/u1, alpha/(alpha^2+beta^2), beta/(alpha^2+beta^2) of RADAU5, evaluated once in extended precision
constexpr double U1 = 3.637834252744495732, ALPH = 2.681082873627752134, BETA = 3.050430199247410569;
constexpr double T11 = 9.1232394870892942792e-02, T12 = -0.14125529502095420843, T13 = -3.0029194105147424492e-02;
constexpr double T21 = 0.24171793270710701896, T22 = 0.20412935229379993199, T23 = 0.38294211275726193779;
constexpr double T31 = 0.96604818261509293619;
constexpr double TI11 = 4.3255798900631553510, TI12 = 0.33919925181580986954, TI13 = 0.54177053993587487119;
constexpr double TI21 = -4.1787185915519047273, TI22 = -0.32768282076106238708, TI23 = 0.47662355450055045196;
constexpr double TI31 = -0.50287263494578687595, TI32 = 2.5719269498556054292, TI33 = -0.59603920482822492497;
}  // namespace rk

struct RadauParams {
    double t_end, rtol, atol, h0;
    int max_steps, newton_max;
    int fd_jacobian;                // 1: CVODE-style difference-quotient Jacobian (R13)
    int fixed_steps;                // > 0: that many equal steps, no error control
    double rtol_t, atol_t, fnewt;   // RADAU5's transformed tolerances and Newton stopping level (R8), set on the host
    double inv_fnewt, inv_n, inv_3n; // 1/fnewt, 1/N, 1/(3N): host-side divisions for the warp path
};

struct RadauResult {
    int status, nstep, naccpt, nrejct, nfcn, njac, ndec, nsol, nnewt_fail;
    double h_last;
};

}  // namespace chem

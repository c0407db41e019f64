// chem.cu -- C ABI (include/chem.h): mechanism compiler, kernels, launch logic.
// sm_100a only; no CPU fallback: every compute entry point fails with CHEM_E_CUDA without a device.
#include "chem_host.h"
#include "chem_radau_warp.cuh"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

using namespace chem;

namespace chem_host {

thread_local std::string g_err;
std::atomic<int64_t> g_launches{0};

int fail(int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return code;
}

// Stream-ordered scratch from a memory pool of the library's own, one per device (created on first use with that device
// current, release threshold lifted so that the blocks of one launch are reused by the next without going back to the
// driver).  The device's default pool -- the host application's -- is left as it is.  chem_scratch_trim gives the cached
// blocks back.
namespace {
constexpr int kMaxPoolDev = 64;
std::mutex g_pool_mu;
cudaMemPool_t g_pool[kMaxPoolDev] = {};
}  // namespace

int scratch_pool(cudaMemPool_t *pool)
{
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxPoolDev) return fail(CHEM_E_UNSUPPORTED, "device ordinal %d not supported (max %d)", dev, kMaxPoolDev - 1);
    std::lock_guard<std::mutex> lock(g_pool_mu);
    if (!g_pool[dev]) {
        cudaMemPoolProps props{};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t p = nullptr;
        CUDA_TRY(cudaMemPoolCreate(&p, &props));
        uint64_t keep = UINT64_MAX;
        const cudaError_t e = cudaMemPoolSetAttribute(p, cudaMemPoolAttrReleaseThreshold, &keep);
        if (e != cudaSuccess) { cudaMemPoolDestroy(p); return fail(CHEM_E_CUDA, "cudaMemPoolSetAttribute: %s", cudaGetErrorString(e)); }
        g_pool[dev] = p;
    }
    *pool = g_pool[dev];
    return CHEM_OK;
}

int scratch_alloc(void **p, size_t bytes, cudaStream_t st)
{
    *p = nullptr;
    cudaMemPool_t pool = nullptr;
    const int rc = scratch_pool(&pool);
    if (rc) return rc;
    CUDA_TRY(cudaMallocFromPoolAsync(p, bytes, pool, st));
    return CHEM_OK;
}
void scratch_free(void *p, cudaStream_t st)
{
    if (p) cudaFreeAsync(p, st);
}
// cached blocks of the current device's pool back to the driver (blocks still in use by queued work stay)
int scratch_trim()
{
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxPoolDev) return CHEM_OK;
    std::lock_guard<std::mutex> lock(g_pool_mu);
    if (g_pool[dev]) CUDA_TRY(cudaMemPoolTrimTo(g_pool[dev], 0));
    return CHEM_OK;
}

}  // namespace chem_host

using chem_host::fail;
using chem_host::g_launches;

#include "chem_fast.inl"

// ------------------------------------------------------------------------------------------------
// Mechanism compiler: validate the description and pack it into coefficient-major / slot-major tables.
extern "C" int chem_mech_load(const chem_mech_desc *d, chem_mech **out)
{
    if (!d || !out) return fail(CHEM_E_ARG, "null argument");
    *out = nullptr;
    const int ns = d->n_species, nr = d->n_reactions;
    if (ns < 2 || nr < 1) return fail(CHEM_E_ARG, "need n_species >= 2 and n_reactions >= 1");
    if (!d->mol_weight || !d->nasa_lo || !d->nasa_hi || !d->nasa_tmid || !d->rxn_type || !d->reac_ptr || !d->reac_sp ||
        !d->reac_nu || !d->prod_ptr || !d->prod_sp || !d->prod_nu || !d->arr_A || !d->arr_b || !d->arr_Ea || !d->eff_ptr)
        return fail(CHEM_E_ARG, "null array in description");
    for (int k = 0; k < ns; k++)
        if (!(d->mol_weight[k] > 0.0) || !(d->nasa_tmid[k] > 0.0)) return fail(CHEM_E_ARG, "species %d: bad weight or tmid", k);

    std::vector<double> W(ns), invW(ns), lo(7 * ns), hi(7 * ns), tmid(ns);
    for (int k = 0; k < ns; k++) {
        W[k] = d->mol_weight[k];
        invW[k] = 1.0 / W[k];
        tmid[k] = d->nasa_tmid[k];
        for (int c = 0; c < 7; c++) {
            lo[c * ns + k] = d->nasa_lo[7 * k + c];
            hi[c * ns + k] = d->nasa_hi[7 * k + c];
        }
    }
    std::vector<int> rtype(nr), slot_sp(6 * nr, 0), slot_nu(6 * nr, 0), eff_ptr(nr + 1, 0), eff_sp;
    std::vector<double> lnA(nr), b(nr), Ta(nr), lnA0(nr, 0.0), b0(nr, 0.0), Ta0(nr, 0.0), dnu(nr), troe(4 * nr, 1.0), eff_dv;
    std::vector<std::vector<std::pair<int, double>>> inc(ns);
    long n_slots_used = 0, n_eff = 0, n_fall = 0, n_troe = 0, n_tb = 0;
    // Table order: reactions sorted by type, the most expensive first (Troe, Lindemann, three-body, elementary; stable),
    // so that the lanes of a warp that evaluate 32 consecutive reactions follow the same branch, and so that the first
    // n_solo (falloff) reactions can be given a thread of their own (see n_solo below).
    std::vector<int> order(nr);
    for (int i = 0; i < nr; i++) {
        if (d->rxn_type[i] < 0 || d->rxn_type[i] > 3) return fail(CHEM_E_ARG, "reaction %d: unknown type %d", i, d->rxn_type[i]);
        order[i] = i;
    }
    std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return d->rxn_type[x] > d->rxn_type[y]; });
    for (int i = 0; i < nr; i++) {
        const int si = order[i];              // source reaction of table slot i
        const int ty = d->rxn_type[si];
        if (ty < 0 || ty > 3) return fail(CHEM_E_ARG, "reaction %d: unknown type %d", i, ty);
        rtype[i] = ty;
        if (!(d->arr_A[si] > 0.0)) return fail(CHEM_E_ARG, "reaction %d: A must be positive", i);
        lnA[i] = std::log(d->arr_A[si]);
        b[i] = d->arr_b[si];
        Ta[i] = d->arr_Ea[si] / kRcal;
        if (ty >= 2) {
            if (!d->low_A || !d->low_b || !d->low_Ea || !(d->low_A[si] > 0.0))
                return fail(CHEM_E_ARG, "reaction %d: falloff needs a positive low-pressure A", i);
            lnA0[i] = std::log(d->low_A[si]);
            b0[i] = d->low_b[si];
            Ta0[i] = d->low_Ea[si] / kRcal;
            n_fall++;
        }
        if (ty == 3) {
            if (!d->troe) return fail(CHEM_E_ARG, "reaction %d: Troe parameters missing", i);
            for (int c = 0; c < 4; c++) troe[c * nr + i] = d->troe[4 * si + c];
            if (troe[nr + i] == 0.0 || troe[2 * nr + i] == 0.0) return fail(CHEM_E_ARG, "reaction %d: Troe T*** or T* is zero", i);
            n_troe++;
        }
        if (ty != 0) n_tb++;
        std::vector<double> net(ns, 0.0);
        double dn = 0.0;
        for (int side = 0; side < 2; side++) {
            const int32_t *ptr = side ? d->prod_ptr : d->reac_ptr, *sp = side ? d->prod_sp : d->reac_sp, *nu = side ? d->prod_nu : d->reac_nu;
            const int n = ptr[si + 1] - ptr[si];
            if (n < 1 || n > 3) return fail(CHEM_E_UNSUPPORTED, "reaction %d: %d species on one side (1..3 supported)", i, n);
            for (int p = 0; p < n; p++) {
                const int k = sp[ptr[si] + p], v = nu[ptr[si] + p];
                if (k < 0 || k >= ns) return fail(CHEM_E_ARG, "reaction %d: species index %d out of range", i, k);
                if (v < 1 || v > 3) return fail(CHEM_E_UNSUPPORTED, "reaction %d: stoichiometric coefficient %d (1..3 supported)", i, v);
                slot_sp[(side * 3 + p) * nr + i] = k;
                slot_nu[(side * 3 + p) * nr + i] = v;
                net[k] += side ? v : -v;
                dn += side ? v : -v;
                n_slots_used++;
            }
        }
        dnu[i] = dn;
        for (int k = 0; k < ns; k++)
            if (net[k] != 0.0) inc[k].push_back({i, net[k]});
        if (ty != 0) {
            if (d->eff_ptr[si + 1] < d->eff_ptr[si]) return fail(CHEM_E_ARG, "eff_ptr not monotone");
            for (int p = d->eff_ptr[si]; p < d->eff_ptr[si + 1]; p++) {
                if (!d->eff_sp || !d->eff_val) return fail(CHEM_E_ARG, "efficiency arrays missing");
                const int k = d->eff_sp[p];
                if (k < 0 || k >= ns) return fail(CHEM_E_ARG, "reaction %d: efficiency species out of range", i);
                eff_sp.push_back(k);
                eff_dv.push_back(d->eff_val[p] - 1.0);
                n_eff++;
            }
        }
        eff_ptr[i + 1] = (int)eff_sp.size();
    }
    std::vector<int> inc_ptr(ns + 1, 0), inc_rx;
    std::vector<double> inc_nu;
    for (int k = 0; k < ns; k++) {
        for (auto &pr : inc[k]) { inc_rx.push_back(pr.first); inc_nu.push_back(pr.second); }
        inc_ptr[k + 1] = (int)inc_rx.size();
    }
    // ---- balanced schedule of the species-production gather of the stage-batched source term (chem_cta.cuh): species k
    // gets c_k = 2^m adjacent threads of one warp, each summing an equal share of its incidence list; the shares are
    // combined by a fixed butterfly (deterministic).  c_k = the power of two above len_k / target, with the smallest
    // target for which all groups fit into the G threads of a state (G as in group_size(), chem_launch.inl).
    const int G_gather = ns <= 32 ? 32 : 128;
    std::vector<int> gat(4 * G_gather, 0), inc2;
    int gat_steps = -1;                                   // -1: no schedule (more species than threads)
    if (ns <= G_gather) {
        auto groups = [&](int target, std::vector<int> *lg) {
            int tot = 0;
            for (int k = 0; k < ns; k++) {
                const int len = inc_ptr[k + 1] - inc_ptr[k], need = (len + target - 1) / target;
                int m2 = 0;
                while ((1 << m2) < need && m2 < 5) m2++;
                if (lg) (*lg)[k] = m2;
                tot += 1 << m2;
            }
            return tot;
        };
        int target = 1;
        while (groups(target, nullptr) > G_gather) target++;
        std::vector<int> lg(ns, 0), ord(ns);
        groups(target, &lg);
        for (int k = 0; k < ns; k++) ord[k] = k;
        std::stable_sort(ord.begin(), ord.end(), [&](int a, int b2) { return lg[a] > lg[b2]; });   // big groups first: aligned starts
        for (int t2 = 0; t2 < G_gather; t2++) gat[4 * t2] = -1;
        int t2 = 0;
        gat_steps = 0;
        for (int k : ord) {
            const int c = 1 << lg[k], len = inc_ptr[k + 1] - inc_ptr[k];
            for (int j = 0; j < c; j++, t2++) {
                gat[4 * t2] = k;
                gat[4 * t2 + 1] = inc_ptr[k] + (int)((long long)len * j / c);
                gat[4 * t2 + 2] = inc_ptr[k] + (int)((long long)len * (j + 1) / c);
                gat[4 * t2 + 3] = lg[k];
            }
            if (lg[k] > gat_steps) gat_steps = lg[k];
        }
    }
    // ---- reaction loop balance of the group kernels: thread t < n_solo evaluates table reaction t only (a Troe reaction
    // costs six exps against two for an elementary one), the other G - n_solo threads stride over the rest; n_solo
    // minimises the heaviest thread under the cost model exps + 0.25 per third-body efficiency
    int n_solo = 0;
    {
        std::vector<double> cost(nr);
        for (int i = 0; i < nr; i++) {
            const double base = rtype[i] == 3 ? 6.0 : (rtype[i] == 2 ? 3.0 : 2.0);
            cost[i] = base + (rtype[i] != 0 ? 0.5 + 0.25 * (eff_ptr[i + 1] - eff_ptr[i]) : 0.0);
        }
        double best = 1e300;
        const int n_heavy = (int)(n_fall < G_gather - 1 ? n_fall : G_gather - 1);
        for (int sN = 0; sN <= n_heavy; sN++) {
            std::vector<double> load(G_gather - sN, 0.0);
            for (int i = sN; i < nr; i++) load[(i - sN) % (G_gather - sN)] += cost[i];
            double mx = sN > 0 ? cost[0] : 0.0;
            for (double v : load) mx = std::max(mx, v);
            if (mx < best - 1e-12) { best = mx; n_solo = sN; }
        }
    }
    for (size_t e = 0; e < inc_rx.size(); e++) { inc2.push_back(inc_rx[e]); inc2.push_back((int)inc_nu[e]); }
    // ---- balanced row gather of the analytical Jacobian (jacobian<128>, chem_device.cuh): the same kind of schedule for
    // as many threads as private rows of N + 3 doubles fit into the matrix storage that is dead during the Jacobian
    // (E1 and the part of the E2 region in front of the slot derivatives: work_doubles / carve, chem_radau.cuh), and one
    // packed record per incidence
    std::vector<int> gatj(4, 0), jinc(8, 0);
    int gatj_T = 0;
    if (ns > 32 && ns <= 128) {
        const size_t e2 = (size_t)2 * ns * (ns + 1) > (size_t)8 * nr ? (size_t)2 * ns * (ns + 1) : (size_t)8 * nr;
        const size_t pool = (size_t)ns * (ns + 1) + e2 - (size_t)8 * nr;
        int T = (int)std::min<size_t>(128, pool / (ns + 3));
        if (T >= ns) {
            auto groups = [&](int target, std::vector<int> *lg) {
                int tot = 0;
                for (int k = 0; k < ns; k++) {
                    const int len = inc_ptr[k + 1] - inc_ptr[k], need = (len + target - 1) / target;
                    int m2 = 0;
                    while ((1 << m2) < need && m2 < 5) m2++;
                    if (lg) (*lg)[k] = m2;
                    tot += 1 << m2;
                }
                return tot;
            };
            int target = 1;
            while (groups(target, nullptr) > T) target++;
            std::vector<int> lg(ns, 0), ord(ns);
            groups(target, &lg);
            for (int k = 0; k < ns; k++) ord[k] = k;
            std::stable_sort(ord.begin(), ord.end(), [&](int a, int b2) { return lg[a] > lg[b2]; });   // big groups first: aligned starts
            gatj.assign(4 * T, 0);
            for (int t2 = 0; t2 < T; t2++) gatj[4 * t2] = -1;
            int t2 = 0;
            for (int k : ord) {
                const int c = 1 << lg[k], len = inc_ptr[k + 1] - inc_ptr[k];
                for (int j = 0; j < c; j++, t2++) {
                    gatj[4 * t2] = k;
                    gatj[4 * t2 + 1] = inc_ptr[k] + (int)((long long)len * j / c);
                    gatj[4 * t2 + 2] = inc_ptr[k] + (int)((long long)len * (j + 1) / c);
                    gatj[4 * t2 + 3] = lg[k];
                }
            }
            gatj_T = T;
            jinc.assign(8 * std::max<size_t>(inc_rx.size(), 1), 0);
            for (size_t e = 0; e < inc_rx.size(); e++) {
                const int i = inc_rx[e];
                jinc[8 * e] = i;
                jinc[8 * e + 1] = (int)inc_nu[e];
                jinc[8 * e + 2] = slot_sp[i] | (slot_sp[nr + i] << 8) | (slot_sp[2 * nr + i] << 16);
                jinc[8 * e + 3] = slot_sp[3 * nr + i] | (slot_sp[4 * nr + i] << 8) | (slot_sp[5 * nr + i] << 16);
                jinc[8 * e + 4] = rtype[i] != 0 ? eff_ptr[i] : 0;
                jinc[8 * e + 5] = rtype[i] != 0 ? eff_ptr[i + 1] : 0;
                jinc[8 * e + 6] = rtype[i] != 0;
            }
        }
    }
    if (eff_sp.empty()) { eff_sp.push_back(0); eff_dv.push_back(0.0); }
    if (inc_rx.empty()) { inc_rx.push_back(0); inc_nu.push_back(0.0); }
    if (inc2.empty()) { inc2.push_back(0); inc2.push_back(0); }

    // ---- exp-job tables for the stage-batched source term of the group kernels (chem_cta.cuh); same idea as
    // chem_fast.inl: k_f, k_r (ln K_c folded in from the NASA coefficients), k_0/k_inf and the three Troe terms are all
    // exp(c0 + c1 lnT + c2/T + c3 T + c4 T^2 + c5 T^3 + c6 T^4).  Job order: [0,nr) k_f, [nr,2nr) k_r, then extras.
    // Eligible when: one common T_mid, <= 63 species, at most three concentration factors per side, 0 < alpha < 1.
    std::vector<double> job_lo, job_hi;
    std::vector<int> rdesc(8 * nr, 0);
    int n_fo = 0, n_jobs = 0, jobs_ok = (ns <= 63);
    for (int k = 1; k < ns; k++) jobs_ok &= (tmid[k] == tmid[0]);
    if (jobs_ok) {
        n_jobs = 2 * nr;
        for (int i = 0; i < nr; i++) n_jobs += (rtype[i] >= 2) + 3 * (rtype[i] == 3);
        job_lo.assign((size_t)n_jobs * 8, 0.0);
        job_hi.assign((size_t)n_jobs * 8, 0.0);
        const double lnPR = std::log(kPatm / kRerg);
        int next_extra = 2 * nr;
        for (int i = 0; i < nr && jobs_ok; i++) {
            int f[6] = {63, 63, 63, 63, 63, 63};
            for (int side = 0; side < 2; side++) {
                int sl = 3 * side;
                for (int p = 0; p < 3; p++)
                    for (int rep = 0; rep < slot_nu[(3 * side + p) * nr + i]; rep++) {
                        if (sl >= 3 * side + 3) { jobs_ok = 0; break; }
                        f[sl++] = slot_sp[(3 * side + p) * nr + i];
                    }
            }
            rdesc[8 * i + 0] = f[0] | (f[1] << 8) | (f[2] << 16);
            rdesc[8 * i + 1] = f[3] | (f[4] << 8) | (f[5] << 16);
            rdesc[8 * i + 2] = rtype[i];
            rdesc[8 * i + 5] = eff_ptr[i];
            rdesc[8 * i + 6] = eff_ptr[i + 1];
            for (int r = 0; r < 2; r++) {
                std::vector<double> &job = r ? job_hi : job_lo;
                const std::vector<double> &na = r ? hi : lo;     // coefficient-major [7][ns]
                double *kf = &job[(size_t)i * 8], *kr = &job[(size_t)(nr + i) * 8];
                kf[0] = lnA[i]; kf[1] = b[i]; kf[2] = -Ta[i];
                double g[7] = {0, 0, 0, 0, 0, 0, 0};
                for (int sl = 0; sl < 6; sl++) {
                    const double v = (sl < 3 ? -1.0 : 1.0) * slot_nu[sl * nr + i];
                    const int k = slot_sp[sl * nr + i];
                    if (v == 0.0) continue;
                    g[0] += v * (na[0 * ns + k] - na[6 * ns + k]);
                    g[1] += v * (-na[0 * ns + k]);
                    g[2] += v * na[5 * ns + k];
                    g[3] += v * (-na[1 * ns + k] / 2.0);
                    g[4] += v * (-na[2 * ns + k] / 6.0);
                    g[5] += v * (-na[3 * ns + k] / 12.0);
                    g[6] += v * (-na[4 * ns + k] / 20.0);
                }
                kr[0] = lnA[i] - dnu[i] * lnPR + g[0];
                kr[1] = b[i] + dnu[i] + g[1];
                kr[2] = -Ta[i] + g[2];
                kr[3] = g[3]; kr[4] = g[4]; kr[5] = g[5]; kr[6] = g[6];
                if (rtype[i] >= 2) {
                    double *c = &job[(size_t)next_extra * 8];
                    c[0] = lnA0[i] - lnA[i]; c[1] = b0[i] - b[i]; c[2] = -(Ta0[i] - Ta[i]);
                }
                if (rtype[i] == 3) {
                    const double al = troe[i], T3 = troe[nr + i], T1 = troe[2 * nr + i], T2 = troe[3 * nr + i];
                    if (!(al > 0.0 && al < 1.0)) { jobs_ok = 0; break; }
                    double *c = &job[(size_t)(next_extra + 1) * 8];
                    c[0] = std::log(1.0 - al); c[3] = -1.0 / T3;
                    c[8] = std::log(al); c[8 + 3] = -1.0 / T1;
                    c[16 + 2] = -T2;
                }
            }
            if (rtype[i] >= 2) {
                rdesc[8 * i + 3] = next_extra;          // k0/kinf job; Troe terms follow at +1..+3
                rdesc[8 * i + 4] = n_fo++;              // falloff ordinal
                next_extra += 1 + 3 * (rtype[i] == 3);
            }
        }
    }
    if (!jobs_ok) { job_lo.assign(8, 0.0); job_hi.assign(8, 0.0); n_jobs = 0; n_fo = 0; }

    int dev = 0, n_sm = 0, optin = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    CUDA_TRY(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));

    // one blob: doubles first, then ints (each array 16-byte aligned)
    std::vector<std::pair<const void *, size_t>> parts;
    std::vector<size_t> offs;
    size_t total = 0;
    auto add = [&](const void *p, size_t bytes) {
        offs.push_back(total);
        parts.push_back({p, bytes});
        total += (bytes + 15) & ~size_t(15);
    };
    add(W.data(), ns * 8); add(invW.data(), ns * 8); add(lo.data(), 7 * ns * 8); add(hi.data(), 7 * ns * 8); add(tmid.data(), ns * 8);
    add(lnA.data(), nr * 8); add(b.data(), nr * 8); add(Ta.data(), nr * 8); add(lnA0.data(), nr * 8); add(b0.data(), nr * 8);
    add(Ta0.data(), nr * 8); add(dnu.data(), nr * 8); add(troe.data(), 4 * nr * 8);
    add(eff_dv.data(), eff_dv.size() * 8); add(inc_nu.data(), inc_nu.size() * 8);
    add(job_lo.data(), job_lo.size() * 8); add(job_hi.data(), job_hi.size() * 8);
    add(rtype.data(), nr * 4); add(slot_sp.data(), 6 * nr * 4); add(slot_nu.data(), 6 * nr * 4);
    add(eff_ptr.data(), (nr + 1) * 4); add(eff_sp.data(), eff_sp.size() * 4);
    add(inc_ptr.data(), (ns + 1) * 4); add(inc_rx.data(), inc_rx.size() * 4); add(rdesc.data(), rdesc.size() * 4);
    add(gat.data(), gat.size() * 4); add(inc2.data(), inc2.size() * 4); add(gatj.data(), gatj.size() * 4); add(jinc.data(), jinc.size() * 4);
    std::vector<char> host(total, 0);
    for (size_t a = 0; a < parts.size(); a++) std::memcpy(host.data() + offs[a], parts[a].first, parts[a].second);

    chem_mech *m = new (std::nothrow) chem_mech;
    if (!m) return fail(CHEM_E_NOMEM, "out of host memory");
    if (cudaMalloc(&m->dev_blob, total) != cudaSuccess) {
        cudaError_t e = cudaGetLastError();
        delete m;
        return fail(CHEM_E_CUDA, "cudaMalloc: %s", cudaGetErrorString(e));
    }
    if (cudaMemcpy(m->dev_blob, host.data(), total, cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaError_t e = cudaGetLastError();
        cudaFree(m->dev_blob);
        delete m;
        return fail(CHEM_E_CUDA, "cudaMemcpy: %s", cudaGetErrorString(e));
    }
    const char *base = static_cast<const char *>(m->dev_blob);
    int a = 0;
    auto D = [&]() { return reinterpret_cast<const double *>(base + offs[a++]); };
    auto I = [&]() { return reinterpret_cast<const int *>(base + offs[a++]); };
    Tables &t = m->t;
    t.n_sp = ns; t.n_rx = nr;
    t.W = D(); t.invW = D(); t.nasa_lo = D(); t.nasa_hi = D(); t.tmid = D();
    t.lnA = D(); t.b = D(); t.Ta = D(); t.lnA0 = D(); t.b0 = D(); t.Ta0 = D(); t.dnu = D(); t.troe = D();
    t.eff_dv = D(); t.inc_nu = D(); t.job_lo = D(); t.job_hi = D();
    t.rtype = I(); t.slot_sp = I(); t.slot_nu = I(); t.eff_ptr = I(); t.eff_sp = I(); t.inc_ptr = I(); t.inc_rx = I(); t.rdesc = I();
    t.gat = reinterpret_cast<const int4 *>(I()); t.inc2 = reinterpret_cast<const int2 *>(I()); t.gat_steps = gat_steps; t.n_solo = n_solo;
    t.gatj = reinterpret_cast<const int4 *>(I()); t.jinc = reinterpret_cast<const int4 *>(I()); t.gatj_T = gatj_T;
    t.n_jobs = n_jobs; t.n_fo = n_fo; t.tmid0 = tmid[0];
    m->n_sm = n_sm;
    m->max_smem_optin = optin;

    // Algorithmic flop model: +,-,*,/ count 1; exp/log/pow/log10/exp10/sqrt count kTrans each:
    // 20 in flops[] (chem_flop_model, the roofline convention), 1 in flops_t1[] (chem_flop_model_t1, for the reader who
    // wants the fraction without that convention).
    auto flop_model = [&](double kTrans, double *fl) {
        const double N = ns;
        const double thermo = ns * (8.0 + 11.0 + 12.0 + 1.0) + kTrans;                      // cp, h, s (Horner), g; one log T
        const double front = 4.0 * ns + 6.0 + ns * 2.0;                                      // closure, Wbar, rho, C_k
        const double rx = nr * (5.0 + 2.0 * kTrans + 4.0 + 3.0) + n_slots_used * 3.0        // ln kf, Kc, 2 exp, products, q
                          + n_tb * 2.0 + n_eff * 2.0 + n_fall * (8.0 + kTrans) + n_troe * (25.0 + 5.0 * kTrans);
        const double wd = 2.0 * inc_rx.size() + 6.0 * ns + 4.0;                              // wdot gather, Tdot, Ydot
        fl[0] = thermo + front + rx + wd + 2.0 * kTrans;
        fl[1] = fl[0] + ns * 7.0 + nr * 40.0 + n_troe * 40.0 + 12.0 * inc_rx.size() + 2.0 * n_eff * 3.0
                + ns * (2.0 * N + 6.0 * N) + N * (2.0 * N + 6.0 * N);                       // derivative slots, rows, columns
        fl[2] = (2.0 / 3.0) * N * N * N * 5.0 + 3.0 * N * N;                                 // real LU + complex LU (4x) + forming E1, E2
        fl[3] = 2.0 * N * N * 5.0 + N * (15.0 + 9.0 + 15.0 + 9.0 + 3.0);                     // real + complex solves, transforms, norm
        fl[4] = 2.0 * N * N + N * 10.0;                                                      // error estimate: one real solve + norm
    };
    flop_model(20.0, m->flops);
    flop_model(1.0, m->flops_t1);
    const int rcf = build_fast(d, m);
    if (rcf != CHEM_OK) { chem_mech_free(m); return rcf; }
    *out = m;
    return CHEM_OK;
}

extern "C" int chem_scratch_trim(void) { return chem_host::scratch_trim(); }

extern "C" void chem_mech_free(chem_mech *m)
{
    if (!m) return;
    chem_host::scratch_trim();      // the launch scratch cached for this device goes back to the driver with the mechanism
    if (m->dev_blob) cudaFree(m->dev_blob);
    if (m->fast_blob) cudaFree(m->fast_blob);
    for (int i = 0; i < 2; i++)
        if (m->hs[i]) cudaStreamDestroy(m->hs[i]);
    delete m;
}

extern "C" int chem_mech_info(const chem_mech *m, int32_t *n_species, int32_t *n_reactions)
{
    if (!m) return fail(CHEM_E_ARG, "null mechanism");
    if (n_species) *n_species = m->t.n_sp;
    if (n_reactions) *n_reactions = m->t.n_rx;
    return CHEM_OK;
}

extern "C" int chem_flop_model(const chem_mech *m, double out[5])
{
    if (!m || !out) return fail(CHEM_E_ARG, "null argument");
    for (int i = 0; i < 5; i++) out[i] = m->flops[i];
    return CHEM_OK;
}

extern "C" int chem_flop_model_t1(const chem_mech *m, double out[5])
{
    if (!m || !out) return fail(CHEM_E_ARG, "null argument");
    for (int i = 0; i < 5; i++) out[i] = m->flops_t1[i];
    return CHEM_OK;
}

extern "C" int64_t chem_launch_count(void) { return g_launches.load(); }
extern "C" const char *chem_last_error(void) { return chem_host::g_err.c_str(); }

#include "chem_kernels.inl"

// ------------------------------------------------------------------------------------------------ no-allocation entry point
// chem_integrate_noalloc (include/chem.h): the shared-memory integration kernels of chem_kernels.inl, launched with their
// global scratch -- the work-queue head and, when the caller asks for cost ordering, the start order -- in a fixed array
// that is part of the library image instead of a block from the stream-ordered allocator.  It is for hosts whose device
// memory is not theirs to ask for at call time: a flow solver or a training framework that took the whole card for its
// own arena at start-up (cudaMallocAsync then fails or makes that arena give memory back), a process held to a hard
// memory budget on a shared or partitioned card, a time-critical loop in which an allocator call that may take a driver
// lock or synchronise the device is not acceptable.  Everything below uses memory that exists from the moment the
// library is loaded: no cudaMalloc / cudaMallocAsync / cudaFree, no cub, no memory pool.
//
// The array: kNoAllocBytes (4 MiB + 4352 B) on EVERY device that loads libchem.so, held until the process exits, whether
// or not this entry point is ever called.  Layout: [0, 256) queue head (one int), [256, 4352) 1024 bucket counters of the
// ordering pass, [4352, ...) start order, one int per state -- hence the limit CHEM_NOALLOC_MAX_STATES per call.
// All calls on one device share it and it keeps whatever the last call left there: each call zeroes the head (and the
// counters when it orders) on its own stream before it launches, and two calls that overlap in time on the GPU
// (different streams, or different host threads without a common stream) corrupt each other's queue.
namespace {

constexpr int kNoAllocBuckets = 1024;
constexpr size_t kNoAllocHeadBytes = 256;
constexpr size_t kNoAllocOrderOff = kNoAllocHeadBytes + kNoAllocBuckets * sizeof(unsigned);   // 4352 = 17 x 256
constexpr size_t kNoAllocBytes = kNoAllocOrderOff + (size_t)CHEM_NOALLOC_MAX_STATES * sizeof(int);

static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocBytes];

// In host code the name g_noalloc_scratch is only a handle for the runtime (a host-side shadow object), NOT the device
// address: handing it to a kernel would make the kernel read and write unrelated memory.  The address is looked up once
// per device, with that device current, and cached.
constexpr int kNoAllocMaxDev = 64;
std::mutex g_noalloc_mu;
void *g_noalloc_ptr[kNoAllocMaxDev] = {};

int noalloc_scratch_ptr(unsigned char **p)
{
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kNoAllocMaxDev) return fail(CHEM_E_UNSUPPORTED, "chem_integrate_noalloc: device ordinal %d not supported (max %d)", dev, kNoAllocMaxDev - 1);
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_ptr[dev]) {
        void *q = nullptr;
        CUDA_TRY(cudaGetSymbolAddress(&q, g_noalloc_scratch));
        if (!q) return fail(CHEM_E_CUDA, "chem_integrate_noalloc: no device address for the scratch array on device %d", dev);
        g_noalloc_ptr[dev] = q;
    }
    *p = static_cast<unsigned char *>(g_noalloc_ptr[dev]);
    return CHEM_OK;
}

// Start order by decreasing cost without a sort library: a counting sort over 1024 cost classes (costs are internal step
// counts; anything above 1023 shares the first class).  Bucket 0 holds the most expensive states.  The order inside a
// class depends on the timing of the atomics; results do not depend on the order at all (it only decides WHEN a state
// starts), so that is harmless.  Equal keys inside a warp are combined into one atomic.
__device__ __forceinline__ int noalloc_bucket(int32_t c)
{
    c = c < 0 ? 0 : (c > kNoAllocBuckets - 1 ? kNoAllocBuckets - 1 : c);
    return kNoAllocBuckets - 1 - c;
}

__global__ void __launch_bounds__(256) noalloc_count_kernel(int n, const int32_t *__restrict__ cost, unsigned *bucket)
{
    const int i = blockIdx.x * 256 + threadIdx.x;
    const int b = i < n ? noalloc_bucket(cost[i]) : kNoAllocBuckets;        // kNoAllocBuckets: lane without a state
    const unsigned peers = __match_any_sync(0xffffffffu, b);
    if (i < n && (int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(&bucket[b], (unsigned)__popc(peers));
}

__global__ void __launch_bounds__(kNoAllocBuckets) noalloc_offsets_kernel(unsigned *bucket)   // one CTA: counts -> first slots
{
    __shared__ unsigned s[kNoAllocBuckets];
    const int t = threadIdx.x;
    const unsigned mine = bucket[t];
    s[t] = mine;
    __syncthreads();
    for (int d = 1; d < kNoAllocBuckets; d <<= 1) {
        const unsigned v = t >= d ? s[t - d] : 0u;
        __syncthreads();
        s[t] += v;
        __syncthreads();
    }
    bucket[t] = s[t] - mine;
}

__global__ void __launch_bounds__(256) noalloc_place_kernel(int n, const int32_t *__restrict__ cost, unsigned *bucket, int *order)
{
    const int i = blockIdx.x * 256 + threadIdx.x, lane = threadIdx.x & 31;
    const int b = i < n ? noalloc_bucket(cost[i]) : kNoAllocBuckets;
    const unsigned peers = __match_any_sync(0xffffffffu, b);
    const int leader = __ffs(peers) - 1;
    unsigned base = 0;
    if (i < n && lane == leader) base = atomicAdd(&bucket[b], (unsigned)__popc(peers));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (i < n) order[base + __popc(peers & ((1u << lane) - 1u))] = i;
}

template <int G>
int noalloc_launch_group(const chem_mech *m, int n, double P, const RadauParams &prm, const double *y_in, double *y_out,
                         const chem_opts *o, chem_stats *stats, int *head, const int *order, cudaStream_t st)
{
    const size_t smem = work_doubles(m->t.n_sp, m->t.n_rx, G / 32, m->t.n_fo) * sizeof(double) * (block_of<G>() / G);
    int occ = 0;
    const int rc = configure(integrate_kernel<G>, m, smem, &occ, block_of<G>());
    if (rc) return rc;
    const int gpb = block_of<G>() / G;
    int grid = (n + gpb - 1) / gpb;
    if (grid > m->n_sm * occ) grid = m->n_sm * occ;
    integrate_kernel<G><<<grid, block_of<G>(), smem, st>>>(m->t, n, P, o ? o->P_per_state : nullptr, prm, y_in, y_out, stats, head, order);
    g_launches++;
    CUDA_TRY(cudaGetLastError());
    return CHEM_OK;
}

int noalloc_launch_warp(const chem_mech *m, int n, double P, const RadauParams &prm, const double *y_in, double *y_out,
                        const chem_opts *o, chem_stats *stats, int *head, const int *order, cudaStream_t st)
{
    const int wpb = kWarpBlock / 32;
    const size_t smem = ((size_t)m->fast.blob_doubles + (size_t)wpb * warp_ws_doubles(m->t.n_sp, m->t.n_rx)) * sizeof(double);
    CUDA_TRY(cudaFuncSetAttribute(integrate_warp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, integrate_warp_kernel, kWarpBlock, smem));
    if (occ < 1) return fail(CHEM_E_UNSUPPORTED, "warp kernel does not fit on an SM");
    int grid = (n + wpb - 1) / wpb;
    if (grid > m->n_sm * occ) grid = m->n_sm * occ;
    integrate_warp_kernel<<<grid, kWarpBlock, smem, st>>>(m->t, m->fast, n, P, o ? o->P_per_state : nullptr, prm, y_in, y_out, stats,
                                                          head, order);
    g_launches++;
    CUDA_TRY(cudaGetLastError());
    return CHEM_OK;
}

}  // namespace

extern "C" int chem_integrate_noalloc(const chem_mech *m, int32_t n, double P, double t_end, double rtol, double atol,
                                      const double *y_in, double *y_out, const chem_opts *o, chem_stats *stats, void *stream)
{
    if (!m || n < 0 || (n > 0 && (!y_in || !y_out))) return fail(CHEM_E_ARG, "bad argument");
    if (!(t_end > 0.0) || !(rtol > 0.0) || !(atol > 0.0)) return fail(CHEM_E_ARG, "t_end, rtol and atol must be positive");
    if (o && (o->kernel < 0 || o->kernel > 3)) return fail(CHEM_E_ARG, "chem_opts.kernel must be 0..3");
    if (n > CHEM_NOALLOC_MAX_STATES)
        return fail(CHEM_E_UNSUPPORTED, "chem_integrate_noalloc: n_states = %d is more than the fixed scratch array holds "
                    "(CHEM_NOALLOC_MAX_STATES = %d); split the batch into several calls on one stream", n, CHEM_NOALLOC_MAX_STATES);
    int kernel = o ? o->kernel : 0;
    if (kernel == 3)
        return fail(CHEM_E_UNSUPPORTED, "chem_integrate_noalloc: the thread-per-state kernel needs a per-launch workspace of 7 KB per "
                    "resident state (277 MB) and is not offered without allocation; use kernel 0, 1 or 2");
    if (kernel == 0) kernel = warp_path_available(m) ? 2 : 1;
    if (kernel == 2 && !warp_path_available(m)) return fail(CHEM_E_UNSUPPORTED, "warp-per-state kernel not available for this mechanism");
    if (n == 0) return CHEM_OK;
    RadauParams prm;      // same derived quantities as integrate_impl (chem_launch.inl)
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

    cudaStream_t st = static_cast<cudaStream_t>(stream);
    unsigned char *scratch = nullptr;
    int rc = noalloc_scratch_ptr(&scratch);      // first call on this device: looks the address up (see chem.h)
    if (rc) return rc;
    int *head = reinterpret_cast<int *>(scratch);
    unsigned *bucket = reinterpret_cast<unsigned *>(scratch + kNoAllocHeadBytes);
    int *order = nullptr;
    const bool ordered = o && o->reorder == 1 && o->cost_hint;      // reorder 0 / 2 / -1: no ordering here (the estimate's keys would need scratch of their own)
    // the array still holds the previous call's queue head and counters: clear what this call starts from
    CUDA_TRY(cudaMemsetAsync(scratch, 0, ordered ? kNoAllocOrderOff : kNoAllocHeadBytes, st));
    if (ordered) {
        order = reinterpret_cast<int *>(scratch + kNoAllocOrderOff);
        const int g = (n + 255) / 256;
        noalloc_count_kernel<<<g, 256, 0, st>>>(n, o->cost_hint, bucket);
        noalloc_offsets_kernel<<<1, kNoAllocBuckets, 0, st>>>(bucket);
        noalloc_place_kernel<<<g, 256, 0, st>>>(n, o->cost_hint, bucket, order);
        g_launches += 3;
        CUDA_TRY(cudaGetLastError());
    }
    if (kernel == 2) rc = noalloc_launch_warp(m, n, P, prm, y_in, y_out, o, stats, head, order, st);
    else rc = group_size(m) == 32 ? noalloc_launch_group<32>(m, n, P, prm, y_in, y_out, o, stats, head, order, st)
                                  : noalloc_launch_group<128>(m, n, P, prm, y_in, y_out, o, stats, head, order, st);
    if (rc == CHEM_OK) const_cast<chem_mech *>(m)->last_kernel = kernel;
    return rc;
}

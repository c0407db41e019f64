// chem_fast.inl -- mechanism compiler, part 2: the "exp job" tables of the compact warp-per-state path
// (chem_warp.cuh).  Included by chem.cu after the definition of chem_mech.
//
// Every transcendental of a source-term evaluation becomes  exp(c0 + c1 ln T + c2/T + c3 T + .. + c6 T^4):
//   kf_i      : ln A + b ln T - Ta/T
//   kr_i      : ln kf - ln Kc,  ln Kc = dnu ln(P_atm/(R T)) - sum_k nu_ki (h_k/RT - s_k/R)   (NASA-7 folded in)
//   k0/kinf   : (ln A0 - ln A) + (b0 - b) ln T - (Ta0 - Ta)/T
//   Troe      : (1-alpha) exp(-T/T***), alpha exp(-T/T*), exp(-T**/T)
// and every rate-of-progress product becomes three concentration factors per side (index 31 = unity).
// Eligibility: N_sp <= 16, N_rx <= 32, molecularity <= 3 per side, one common NASA switch temperature, 0 < alpha < 1, and the extra jobs
// (falloff, Troe) fit in the lanes the reactions leave free in two rounds of 32.

namespace {

int build_fast(const chem_mech_desc *d, chem_mech *m)
{
    FastTables &f = m->fast;
    f.enabled = 0;
    const int ns = d->n_species, nr = d->n_reactions;
    if (ns > 16 || nr > 32) return CHEM_OK;
    for (int k = 1; k < ns; k++)
        if (d->nasa_tmid[k] != d->nasa_tmid[0]) return CHEM_OK;
    int extra = 0;
    for (int i = 0; i < nr; i++) {
        if (d->rxn_type[i] >= 2) extra += 1;
        if (d->rxn_type[i] == 3) {
            extra += 3;
            const double al = d->troe[4 * i];
            if (!(al > 0.0 && al < 1.0)) return CHEM_OK;
        }
    }
    if (extra > 2 * (32 - nr)) return CHEM_OK;

    std::vector<double> job[2] = {std::vector<double>(kJobs * kJobW, 0.0), std::vector<double>(kJobs * kJobW, 0.0)};
    std::vector<double> sp[2] = {std::vector<double>(16 * kJobW, 0.0), std::vector<double>(16 * kJobW, 0.0)};
    std::vector<int> slots(32, 0), type(32, -1), jobs(32, 0);
    // unused job rows stay all-zero: they evaluate exp(0) = 1 and are never read
    for (int k = 0; k < ns; k++)
        for (int r = 0; r < 2; r++) {
            const double *a = (r ? d->nasa_hi : d->nasa_lo) + 7 * k;
            for (int c = 0; c < 6; c++) sp[r][k * kJobW + c] = a[c];
            sp[r][k * kJobW + 6] = d->mol_weight[k];
            sp[r][k * kJobW + 7] = 1.0 / d->mol_weight[k];
        }
    int free_slot = nr;   // next spare (round, lane) position: round 0 lanes nr..31, then round 1 lanes nr..31
    auto alloc = [&](int n) -> int {   // n consecutive result slots inside one round, or -1
        for (;;) {
            const int round_end = free_slot < 32 ? 32 : kJobs;
            if (free_slot + n <= round_end) {
                const int s0 = free_slot;
                free_slot += n;
                if (free_slot == 32) free_slot = 32 + nr;
                return s0;
            }
            if (free_slot >= 32) return -1;
            free_slot = 32 + nr;
        }
    };
    const double lnPR = std::log(kPatm / kRerg);
    for (int i = 0; i < nr; i++) {
        const double lnA = std::log(d->arr_A[i]), b = d->arr_b[i], Ta = d->arr_Ea[i] / kRcal;
        type[i] = d->rxn_type[i];
        double dnu = 0.0;
        // concentration factors with multiplicity, three per side, index 31 = unity
        for (int side = 0; side < 2; side++) {
            const int32_t *ptr = side ? d->prod_ptr : d->reac_ptr, *spi = side ? d->prod_sp : d->reac_sp, *nu = side ? d->prod_nu : d->reac_nu;
            int sl = side * 3;
            for (int p = ptr[i]; p < ptr[i + 1]; p++) {
                dnu += side ? nu[p] : -nu[p];
                for (int rep = 0; rep < nu[p]; rep++, sl++) {
                    if (sl >= side * 3 + 3) return CHEM_OK;          // molecularity above 3: not eligible
                    slots[i] |= spi[p] << (5 * sl);
                }
            }
            for (; sl < side * 3 + 3; sl++) slots[i] |= 31 << (5 * sl);
        }
        for (int r = 0; r < 2; r++) {
            double *kf = &job[r][i * kJobW], *kr = &job[r][(32 + i) * kJobW];
            kf[0] = lnA; kf[1] = b; kf[2] = -Ta;
            // sum_k nu_ki g_k with g = a0 (1 - ln T) - a1 T/2 - a2 T^2/6 - a3 T^3/12 - a4 T^4/20 + a5/T - a6
            double g[7] = {0, 0, 0, 0, 0, 0, 0};
            for (int side = 0; side < 2; side++) {
                const int32_t *ptr = side ? d->prod_ptr : d->reac_ptr, *spi = side ? d->prod_sp : d->reac_sp, *nu = side ? d->prod_nu : d->reac_nu;
                for (int p = ptr[i]; p < ptr[i + 1]; p++) {
                    const double v = side ? nu[p] : -nu[p];
                    const double *a = (r ? d->nasa_hi : d->nasa_lo) + 7 * spi[p];
                    g[0] += v * (a[0] - a[6]);
                    g[1] += v * (-a[0]);
                    g[2] += v * a[5];
                    g[3] += v * (-a[1] / 2.0);
                    g[4] += v * (-a[2] / 6.0);
                    g[5] += v * (-a[3] / 12.0);
                    g[6] += v * (-a[4] / 20.0);
                }
            }
            // ln kr = ln kf - dnu (ln(P_atm/R) - ln T) + sum nu g
            kr[0] = lnA - dnu * lnPR + g[0];
            kr[1] = b + dnu + g[1];
            kr[2] = -Ta + g[2];
            kr[3] = g[3]; kr[4] = g[4]; kr[5] = g[5]; kr[6] = g[6];
        }
        if (d->rxn_type[i] >= 2) {
            const int s0 = alloc(1);
            if (s0 < 0) return CHEM_OK;
            for (int r = 0; r < 2; r++) {
                double *c = &job[r][s0 * kJobW];
                c[0] = std::log(d->low_A[i]) - lnA;
                c[1] = d->low_b[i] - b;
                c[2] = -(d->low_Ea[i] / kRcal - Ta);
            }
            jobs[i] = s0;
        }
        if (d->rxn_type[i] == 3) {
            const int s1 = alloc(3), s2 = s1 + 1, s3 = s1 + 2;
            if (s1 < 0) return CHEM_OK;
            const double al = d->troe[4 * i], T3 = d->troe[4 * i + 1], T1 = d->troe[4 * i + 2], T2 = d->troe[4 * i + 3];
            for (int r = 0; r < 2; r++) {
                double *c = &job[r][s1 * kJobW];
                c[0] = std::log(1.0 - al); c[3] = -1.0 / T3;
                c = &job[r][s2 * kJobW];
                c[0] = std::log(al); c[3] = -1.0 / T1;
                c = &job[r][s3 * kJobW];
                c[2] = -T2;
            }
            jobs[i] |= s1 << 8;
        }
    }
    // incidence lists (species -> reactions with net coefficient) and efficiency lists (alpha - 1)
    std::vector<double> inc_nu, eff_dv;
    std::vector<int> inc_rx, eff_sp, desc(32 * 8, 0);
    int n_falloff = 0;
    for (int l = 0; l < 32; l++) {
        desc[8 * l] = slots[l]; desc[8 * l + 2] = type[l]; desc[8 * l + 3] = jobs[l];
        desc[8 * l + 1] = type[l] >= 2 ? n_falloff++ : 0;       // falloff ordinal: phase-2 lane group of warp_rhs3
    }
    if (n_falloff > 5) return CHEM_OK;                          // 6 phase-2 lanes per falloff reaction
    for (int i = 0; i < nr; i++) {
        desc[8 * i + 4] = (int)eff_sp.size();
        if (d->rxn_type[i] != 0)
            for (int p = d->eff_ptr[i]; p < d->eff_ptr[i + 1]; p++) { eff_sp.push_back(d->eff_sp[p]); eff_dv.push_back(d->eff_val[p] - 1.0); }
        desc[8 * i + 5] = (int)eff_sp.size();
    }
    for (int k = 0; k < ns; k++) {
        desc[8 * k + 6] = (int)inc_rx.size();
        for (int i = 0; i < nr; i++) {
            double net = 0.0;
            for (int p = d->reac_ptr[i]; p < d->reac_ptr[i + 1]; p++) if (d->reac_sp[p] == k) net -= d->reac_nu[p];
            for (int p = d->prod_ptr[i]; p < d->prod_ptr[i + 1]; p++) if (d->prod_sp[p] == k) net += d->prod_nu[p];
            if (net != 0.0) { inc_rx.push_back(i); inc_nu.push_back(net); }
        }
        desc[8 * k + 7] = (int)inc_rx.size();
    }
    auto pad2 = [](size_t n) { return (n + 1) & ~size_t(1); };
    const int o_inc_nu = kOffLists, o_eff_dv = o_inc_nu + (int)pad2(inc_nu.size());
    const int o_inc_rx = o_eff_dv + (int)pad2(eff_dv.size()), o_eff_sp = o_inc_rx + (int)pad2(inc_rx.size()) + 2;
    const int total = (int)pad2(o_eff_sp + pad2(eff_sp.size()) / 2 + 1);
    std::vector<double> host(total, 0.0);
    int *hdr = reinterpret_cast<int *>(host.data());
    const int LD = ns | 1;
    hdr[0] = ns; hdr[1] = nr; hdr[2] = o_inc_nu; hdr[3] = o_inc_rx; hdr[4] = o_eff_dv; hdr[5] = o_eff_sp; hdr[6] = LD; hdr[7] = n_falloff;
    std::memcpy(&host[kOffJobLo], job[0].data(), kJobs * kJobW * 8);
    std::memcpy(&host[kOffJobHi], job[1].data(), kJobs * kJobW * 8);
    std::memcpy(&host[kOffSpLo], sp[0].data(), 16 * kJobW * 8);
    std::memcpy(&host[kOffSpHi], sp[1].data(), 16 * kJobW * 8);
    {   // descriptor words as two planes of int4 per lane (conflict-free 16-byte loads)
        int *dst = reinterpret_cast<int *>(&host[kOffDesc]);
        for (int l = 0; l < 32; l++)
            for (int c = 0; c < 8; c++) dst[(c < 4 ? 0 : 128) + 4 * l + (c & 3)] = desc[8 * l + c];
    }
    if (!inc_nu.empty()) std::memcpy(&host[o_inc_nu], inc_nu.data(), inc_nu.size() * 8);
    if (!eff_dv.empty()) std::memcpy(&host[o_eff_dv], eff_dv.data(), eff_dv.size() * 8);
    {   // incidence entries as (reaction, net coefficient) int pairs: one 8-byte load per entry in the kernels
        std::vector<int> pairs(2 * inc_rx.size());
        for (size_t e = 0; e < inc_rx.size(); e++) { pairs[2 * e] = inc_rx[e]; pairs[2 * e + 1] = (int)inc_nu[e]; }
        if (!pairs.empty()) std::memcpy(&host[o_inc_rx], pairs.data(), pairs.size() * 4);
    }
    if (!eff_sp.empty()) std::memcpy(&host[o_eff_sp], eff_sp.data(), eff_sp.size() * 4);
    CUDA_TRY(cudaMalloc(&m->fast_blob, host.size() * 8));
    CUDA_TRY(cudaMemcpy(m->fast_blob, host.data(), host.size() * 8, cudaMemcpyHostToDevice));
    f.blob = static_cast<const double *>(m->fast_blob);
    f.blob_doubles = total;
    f.n_sp = ns; f.n_rx = nr; f.tmid = d->nasa_tmid[0];
    f.enabled = 1;
    return CHEM_OK;
}

}  // namespace

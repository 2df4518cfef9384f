// One exact family (DV, NG) of the fused pass per object file (compiled in parallel by build.py with -DPASS_DV=..
// -DPASS_NG=.. -DPASS_PCAP=.. -DPASS_NAME=..): the launcher PASS_NAME and PASS_NAME_table, which fills the family's
// kernel-parameter table from the generic code tables.
#include "pass_exact.cuh"

#include <cstring>

#if !defined(PASS_DV) || !defined(PASS_NG) || !defined(PASS_PCAP) || !defined(PASS_NAME)
#error "compile with -DPASS_DV=<column degree> -DPASS_NG=<gen edges per column> -DPASS_PCAP=<partner slots per gen edge> -DPASS_NAME=<symbol>"
#endif

#define PASS_CAT2(a, b) a##b
#define PASS_CAT(a, b) PASS_CAT2(a, b)

namespace qc {
using Table = ExactTable<PASS_DV, PASS_NG, PASS_PCAP>;

size_t PASS_CAT(PASS_NAME, _table)(const HostTables& h, void* out) {
    if (!out) return sizeof(Table);
    Table& T = *static_cast<Table*>(out);
    memset(&T, 0, sizeof(Table));
    for (int c = 0; c < h.n_cols && c < kMaxExactCols; ++c) {
        const ColDesc& cd = h.col[c];
        auto& e = T.c[c];
        e.col = cd.col; e.ebeg = cd.ebeg;
        for (int k = 0; k < PASS_DV; ++k) {
            const EdgeDesc& d = h.edge[cd.ebeg + k];
            e.shift[k] = d.shift; e.t_off[k] = d.t_off; e.p_off[k] = d.p_off; e.delta[k] = d.delta;
        }
        for (int g = 0; g < PASS_NG; ++g) {
            const GenDesc& gd = h.gen[cd.gbeg + g];
            e.g_np[g] = gd.np; e.g_counter[g] = gd.counter; e.g_pbeg[g] = cd.pbeg + gd.pbeg;
            for (int j = 0; j < PASS_PCAP; ++j) {
                const bool have = j < gd.np;
                e.g_off[g * PASS_PCAP + j] = have ? h.partner[cd.pbeg + gd.pbeg + j].off : -1;
                e.g_delta[g * PASS_PCAP + j] = have ? h.partner[cd.pbeg + gd.pbeg + j].delta : 0;
            }
        }
    }
    return sizeof(Table);
}

template <int V, bool FINAL>
static void launch_exact(const PassLaunch& L) {
    const bool with_check = !FINAL && L.check_args != nullptr;
    const dim3 grid((L.args.Z + kThreads * V - 1) / (kThreads * V), L.n_cols + (with_check ? 1 : 0), L.n_frames);
    PassArgs args = L.args;
    args.cand_y = with_check ? L.n_cols : -1;
    static const CheckTables no_tab{nullptr, nullptr};
    static const CheckArgs no_args{};
    const CheckTables& ctab = with_check ? *static_cast<const CheckTables*>(L.check_tab) : no_tab;
    const CheckArgs& ca = with_check ? *static_cast<const CheckArgs*>(L.check_args) : no_args;
    if (FINAL)
        k_pass_exact<PASS_DV, PASS_NG, PASS_PCAP, V, FINAL><<<grid, kThreads, 0, L.stream>>>(
            *static_cast<const Table*>(L.exact), args, L.tab.partner, ctab, ca);
    else
        launch_pdl(k_pass_exact<PASS_DV, PASS_NG, PASS_PCAP, V, FINAL>, grid, dim3(kThreads), 0, L.stream,
                   *static_cast<const Table*>(L.exact), args, L.tab.partner, ctab, ca);
}

void PASS_NAME(const PassLaunch& L) {
    if (L.prepare_only) return;                          // no attributes to set: static shared memory only
    if (L.V == 2) { if (L.final_mode) launch_exact<2, true>(L); else launch_exact<2, false>(L); }
    else { if (L.final_mode) launch_exact<1, true>(L); else launch_exact<1, false>(L); }
}
}  // namespace qc

// The frame-interleaved kernel family (pass_il.cuh): batched decodes of codes outside the exact families.
#define QC_IL_IMPL
#include "pass_il.cuh"

namespace qc {

void launch_pass_il_entry(const IlLaunch& L) { launch_pass_il(L); }

void launch_il_init(const PassTables& ptab, const CheckTables& ctab, const IlArgs& a, cudaStream_t st) {
    const int tiles32 = (a.Z + 31) / 32;
    if (a.n_cols > 0) k_il_init_cols<<<dim3(tiles32 * a.n_cols, a.n_groups), 256, 0, st>>>(ptab, a);
    k_il_init_rows<<<dim3(tiles32 * a.mb, a.n_groups), 256, 0, st>>>(ctab, a);
}

void launch_il_cand(const CheckTables& ctab, const CheckArgs& c, const IlArgs& a, int blocks, cudaStream_t st) {
    launch_pdl(k_cand_il, dim3(blocks), dim3(256), 0, st, ctab, c, a);
}

void launch_il_check_final(const CheckTables& ctab, const IlArgs& a, cudaStream_t st) {
    const int tiles32 = (a.Z + 31) / 32;
    k_il_check_final<<<dim3(tiles32 * a.mb, a.n_groups), 256, 0, st>>>(ctab, a);
}

}  // namespace qc

// k_vn_pass -- steps a1 + a2 of the hot path: the fused check-node / variable-node update of one flooding iteration
// (Algorithm 1 steps 2-3), VN-centric, one thread per active variable.
//
// The thread of variable v = (column C, index i) needs, for each of its edges (c,v), the messages of the OTHER edges
// of check c from the previous iteration.  In a pair row that is ONE float (the partner edge) plus the static term
// t_c; both are contiguous cyclic runs in i, so a warp reads 128 contiguous bytes per load (one wrap-around per row).
// Phase 1 issues every such load of the variable back to back (2*dv independent loads in flight per thread: memory
// latency is paid once per variable, not once per edge).  Phase 2 folds the rows with more than one partner (the few
// "top" rows) into one equivalent partner value, while the phase-1 loads are still in flight.  Phase 3 forms every
// m_cv, phase 4 the posterior, the hard decision and every L_vc by prefix/suffix sums, and writes q(L_vc), aligned.
#pragma once

#include "common.cuh"

namespace qc {

template <int DV, bool EXACT, class Tables>
__global__ void __launch_bounds__(kThreads) k_vn_pass(const __grid_constant__ Tables tab, const VnArgs a) {
    const int f = blockIdx.y;
    if (a.done[f]) return;                                   // frame already stopped: its state stays frozen
    const int ca = blockIdx.x / a.tiles;                     // block-uniform active column
    const int tile = blockIdx.x - ca * a.tiles;
    const ColDesc cd = tab.col[ca];
    const int Z = a.Z;
    const int dv = EXACT ? DV : cd.dv;
    const float* __restrict__ qold = a.qold + (int64_t)f * a.EZ;
    float* __restrict__ qnew = a.qnew + (int64_t)f * a.EZ;
    const float* __restrict__ tf = a.t + (int64_t)f * a.m;

    const int ii = tile * kThreads + threadIdx.x;
    const bool valid = ii < Z;
    const int i = valid ? ii : Z - 1;                        // clamp: loads stay in bounds, stores are guarded
    const int64_t v = (int64_t)f * a.n + (int64_t)cd.col * Z + i;
    const float Q = __ldg(a.llr + v);

    // phase 1: all loads of the pair rows
    float tv[DV], qv[DV];
#pragma unroll
    for (int k = 0; k < DV; ++k) {
        tv[k] = 0.0f;
        qv[k] = 0.0f;
        if (EXACT || k < dv) {
            const PairDesc pd = tab.pair[cd.ebeg + k];
            int r = i - pd.shift; r += (r < 0) ? Z : 0;      // check index inside the block row
            tv[k] = __ldg(tf + pd.t_off + r);
            if (pd.p_off >= 0) {
                int ip = i + pd.delta; ip -= (ip >= Z) ? Z : 0;   // partner variable index in its column
                qv[k] = __ldg(qold + pd.p_off + ip);
            }
        }
    }

    // phase 2: rows with 0 or >= 2 partners: fold the partners into one equivalent q (boxplus is associative)
    for (int g = 0; g < cd.ng; ++g) {
        const GenDesc gd = tab.gen[cd.gbeg + g];
        float num = 0.0f, den = 1.0f;
        unsigned sg = 0;
#pragma unroll 4
        for (int j = 0; j < gd.np; ++j) {
            const PartnerDesc pp = tab.partner[gd.pbeg + j];
            int ip = i + pp.delta; ip -= (ip >= Z) ? Z : 0;
            const float qa = __ldg(qold + pp.off + ip);
            sg ^= sign_of(qa);
            boxplus_acc(fabsf(qa), num, den);
        }
        const float qe = with_sign(__fdiv_rn(num, den), sg);
#pragma unroll
        for (int k = 0; k < DV; ++k) qv[k] = (k == gd.k) ? qe : qv[k];
    }

    // phase 3: check-node rule per edge: partner [+] static term, sign product with (-1)^{s_c} inside t
#pragma unroll
    for (int k = 0; k < DV; ++k) {
        const float qa = fabsf(qv[k]), tt = fabsf(tv[k]);
        const float mag = mag_of(qa + tt, fmaf(qa, tt, 1.0f));
        const float m = with_sign(mag, sign_of(qv[k]) ^ sign_of(tv[k]));
        tv[k] = (EXACT || k < dv) ? m : 0.0f;                // tv now holds m_cv
    }

    // phase 4: variable-node rule: L_v = Q_v + sum m; L_vc by direct exclusion (prefix + suffix sums)
    float suf[DV + 1];
    suf[DV] = 0.0f;
#pragma unroll
    for (int k = DV - 1; k >= 0; --k) suf[k] = suf[k + 1] + tv[k];
    float run = Q;
#pragma unroll
    for (int k = 0; k < DV; ++k) {
        const float Lvc = run + suf[k + 1];
        run += tv[k];
        if ((EXACT || k < dv) && valid) qnew[(int64_t)(cd.ebeg + k) * Z + i] = q_of_llr(Lvc);
    }
    if (valid) {
        a.hard[v] = run < 0.0f ? 1 : 0;                      // 0 iff L_v >= 0
        if (a.post) a.post[v] = run;
    }
}

template <int DV, bool EXACT>
void launch_vn(const VnLaunch& L) {
    if (L.inl) k_vn_pass<DV, EXACT, VnTablesInline><<<L.grid, kThreads, 0, L.stream>>>(*L.inl, L.args);
    else k_vn_pass<DV, false, VnTablesGlobal><<<L.grid, kThreads, 0, L.stream>>>(L.glob, L.args);
}

}  // namespace qc

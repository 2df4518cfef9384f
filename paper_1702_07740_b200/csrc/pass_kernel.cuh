// k_pass -- steps a1 + a2 (+ the cheap part of a3) of the hot path: one flooding iteration of Algorithm 1 (steps 2-4,
// P:348-363), fused and VN-centric, for ANY code the handle accepts (active column degree <= kMaxDv, any row degree).
// Codes whose columns all have one of the BASELINE.json shapes run k_pass_exact (pass_exact.cuh: same arithmetic,
// compile-time degrees, tables in the kernel parameters).  One CTA = one tile of kThreads consecutive variables of one
// active column.
//
// The thread of variable v = (column C, index i) needs, for each of its edges (c,v), the messages of the OTHER edges
// of check c from the previous iteration, plus the static term t_c.  Both are cyclic runs in i; thanks to the halo
// behind every run (common.cuh) the window a tile reads is contiguous, so its start is block-uniform: the preamble
// computes it once per edge into shared memory and the per-thread cost of an access is one 64-bit multiply-add.
//   phase 1  loads: t of every row, the partner of every pair row
//   phase 2  gen rows (the rows that are not "two active edges + one absorbed variable"): fold the partners into
//            one equivalent q; the row's counter edge also forms the parity of the PREVIOUS iteration's hard
//            decisions from the bit-0 tags (rows without absorbed variable only: the cheap early-exit filter)
//   phase 3  check-node rule per edge
//   phase 4  variable-node rule: L_v, xhat_v, every L_vc by prefix/suffix sums (direct
//            exclusion, no total-minus-self); writes w(L_vc), aligned and coalesced
// FINAL = true: same arithmetic on each frame's frozen state, writes the outputs (hard bits, posterior) instead.
#pragma once

#include "common.cuh"

namespace qc {

template <bool FINAL>
__global__ void __launch_bounds__(kThreads) k_pass(const PassTables tab, const PassArgs a) {
    __shared__ int2 s_eo[kMaxDv];
    __shared__ GenDesc s_gd[kMaxDv];
    __shared__ int s_po[kMaxPartners];

    pdl_launch();
    pdl_wait();
    const int f = blockIdx.y;
    int in_buf;
    if (FINAL) {
        const int T = a.iters[f];
        if (T <= 0) return;                                  // t = 0: k_init_cols wrote the outputs
        in_buf = (T - 1) % 3;
    } else {
        if (a.done[f]) return;                               // frame already stopped: its state stays frozen
        in_buf = a.in_buf;
    }
    const int ca = blockIdx.x / a.tiles;                     // block-uniform active column
    const int tile = blockIdx.x - ca * a.tiles;
    const ColDesc cd = tab.col[ca];
    const int Z = a.Z, Zs = a.Zs;
    const int dv = cd.dv, ng = cd.ng;
    const int tid = threadIdx.x;
    const int i0 = tile * kThreads;
    const int i = i0 + tid;

    // preamble: window starts of this tile, once per edge
    if (tid < dv) {
        const EdgeDesc d = tab.edge[cd.ebeg + tid];
        int r0 = i0 - d.shift; r0 += (r0 < 0) ? Z : 0;       // check index of the tile's first variable
        int qo = -1;
        if (d.p_off >= 0) { int x = i0 + d.delta; x -= (x >= Z) ? Z : 0; qo = d.p_off + x; }
        s_eo[tid] = make_int2(qo < 0 ? -1 : 4 * qo, 4 * (d.t_off + r0));    // byte offsets
    }
    if (tid < ng) s_gd[tid] = tab.gen[cd.gbeg + tid];
#pragma unroll 1
    for (int j = tid; j < cd.np; j += kThreads) {
        const PartnerDesc p = tab.partner[cd.pbeg + j];
        int x = i0 + p.delta; x -= (x >= Z) ? Z : 0;
        s_po[j] = 4 * (p.off + x);
    }
    __syncthreads();

    const float* __restrict__ qP = a.qb[in_buf] + (int64_t)f * a.EZs + tid;
    const float* __restrict__ tP = a.t + (int64_t)f * a.mZs + tid;
    const bool valid = i < Z;
    const float Q = valid ? llr_to_log2(__ldg(a.llr + (int64_t)f * a.n + (int64_t)cd.col * Z + i)) : 0.0f;
    const unsigned xb = (!FINAL && ng > 0) ? a.hard_in[(int64_t)f * a.AZs + (int64_t)ca * Zs + i] : 0u;

    // phase 1: loads
    float tv[kMaxDv], wv[kMaxDv];
#pragma unroll 1
    for (int k = 0; k < dv; ++k) {
        const int2 o = s_eo[k];
        tv[k] = __ldg(byte_ptr(tP, o.y));
        if (o.x != -1) wv[k] = __ldg(byte_ptr(qP, o.x));
    }

    // phase 2: gen rows: fold the partners into one equivalent q (the rule is associative); bit 0 of a gen edge's
    // state is its variable's hard decision, so the XOR of the raw words carries sign product AND parity
    unsigned bad = 0;
#pragma unroll 1
    for (int g = 0; g < ng; ++g) {
        const GenDesc gd = s_gd[g];
        float num = 0.0f, den = 1.0f;
        unsigned xa = 0u;
#pragma unroll 4
        for (int j = 0; j < gd.np; ++j) {
            const unsigned wb = __float_as_uint(__ldg(byte_ptr(qP, s_po[gd.pbeg + j])));
            xa ^= wb;
            boxplus_acc(__uint_as_float(wb & 0x7ffffffeu), num, den);
        }
        wv[g] = with_sign(num * rcp_approx(den), xa & 0x80000000u);
        if (!FINAL && gd.counter)    // parity of the row at the input iteration: s_c ^ XOR xhat (t = (-1)^{s_c} 0)
            bad |= (xa ^ xb ^ (__float_as_uint(tv[g]) >> 31)) & (valid ? 1u : 0u);
    }

    // phase 3: check-node rule: partner [+] static term; the sign product includes (-1)^{s_c} via t
#pragma unroll 1
    for (int k = 0; k < dv; ++k) {
        const float qa = fabsf(wv[k]), tt = fabsf(tv[k]);
        const float mag = mag_of(qa + tt, fmaf(qa, tt, 1.0f));
        tv[k] = with_sign(mag, sign_of(wv[k]) ^ sign_of(tv[k]));   // tv now holds m'_cv
    }

    // phase 4: variable-node rule
    float suf[kMaxDv + 1];
    suf[dv] = 0.0f;
#pragma unroll 1
    for (int k = dv - 1; k >= 0; --k) suf[k] = suf[k + 1] + tv[k];
    const float L = Q + suf[0];                              // L'_v
    const unsigned xh = __float_as_uint(L) >> 31;            // 0 iff L_v >= 0
    if (FINAL) {
        if (valid) {
            const int64_t vv = (int64_t)f * a.n + (int64_t)cd.col * Z + i;
            a.d_hard[vv] = (uint8_t)xh;
            if (a.d_post) a.d_post[vv] = L * kLn2;
        }
        return;
    }
    a.hard_out[(int64_t)f * a.AZs + (int64_t)ca * Zs + i] = (uint8_t)xh;
    if (ng > 0 && __any_sync(0xffffffffu, bad != 0) && (tid & 31) == 0) a.topbad[f] = 1;

    // tiles that own the first kHalo entries of the run write them twice (run + halo)
    const int nrep = (i0 < kHalo) ? 2 : 1;
#pragma unroll 1
    for (int rep = 0; rep < nrep; ++rep) {
        float* __restrict__ sp = a.qb[a.out_buf] + (int64_t)f * a.EZs + (int64_t)cd.ebeg * Zs + (rep ? Z : 0) + i;
        float run = Q;
#pragma unroll 1
        for (int k = 0; k < dv; ++k) {
            const float Lvc = run + suf[k + 1];              // Q + sum_{k' != k} m_k'
            run += tv[k];
            unsigned wb = __float_as_uint(w_of(Lvc));
            if (k < ng) wb = (wb & 0xfffffffeu) | xh;        // gen edge: tag with the hard decision
            if (valid) *sp = __uint_as_float(wb);
            sp = byte_ptr(sp, 4u * Zs);
        }
    }
}

inline void launch_pass_any(const PassLaunch& L) {
    if (L.final_mode) k_pass<true><<<L.grid, kThreads, 0, L.stream>>>(L.tab, L.args);
    else launch_pdl(k_pass<false>, L.grid, dim3(kThreads), 0, L.stream, L.tab, L.args);
}

}  // namespace qc

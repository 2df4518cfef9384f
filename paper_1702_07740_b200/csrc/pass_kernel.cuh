// k_pass -- steps a1 + a2 (+ the cheap part of a3) of the hot path: one flooding iteration of Algorithm 1 (steps 2-4,
// P:348-363), fused and VN-centric.  One CTA = one tile of kThreads*V consecutive variables of one active column.
//
// The thread of variable v = (column C, index i) needs, for each of its edges (c,v), the messages of the OTHER edges
// of check c from the previous iteration, plus the static term t_c.  Both are cyclic runs in i; thanks to the halo
// behind every run (common.cuh) the window a tile reads is contiguous, so its start is block-uniform: the preamble
// computes it once per edge into shared memory and the per-thread cost of an access is one 64-bit multiply-add.
//   phase 1  every load, back to back: the partners of the gen rows (EXACT: NG x PCAP predicated slots per thread, so
//            that they are in flight together with everything else instead of one dependent round trip per gen
//            edge), t of every row, the partner of every pair row
//   phase 2  gen rows (the few rows that are not "two active edges + one absorbed variable"): fold the partners into
//            one equivalent q; the row's counter edge also forms the parity of the PREVIOUS iteration's hard
//            decisions from the bit-0 tags (rows without absorbed variable only: the cheap early-exit filter)
//   phase 3  check-node rule per edge
//   phase 4  variable-node rule: L_v, xhat_v, every L_vc by prefix/suffix sums (direct
//            exclusion, no total-minus-self); writes w(L_vc), aligned and coalesced
// FINAL = true: same arithmetic on each frame's frozen state, writes the outputs (hard bits, posterior) instead.
#pragma once

#include "common.cuh"

namespace qc {

// EXACT: every active column has DV edges, the first NG of them gen edges; the first PCAP partners of each gen edge
// sit in fixed (compile-time) slots, the rare rest (row degree > PCAP + 1) is folded in a slow loop afterwards.
template <int DV, int NG, int PCAP, bool EXACT, int V, bool FINAL>
__global__ void __launch_bounds__(kThreads) k_pass(const PassTables tab, const PassArgs a) {
    constexpr int UNR = EXACT ? DV : 1;
    constexpr int NGS = NG > 0 ? NG : 1;
    constexpr int UNG = EXACT ? NGS : 1;
    static_assert(!EXACT || NGS * PCAP <= kThreads, "one preamble thread per partner slot");
    __shared__ int2 s_eo[DV];
    __shared__ GenDesc s_gd[NGS];
    __shared__ int s_po[EXACT ? NGS * PCAP : kMaxPartners];

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
    const int dv = EXACT ? DV : cd.dv;
    const int ng = EXACT ? NG : cd.ng;
    const int tid = threadIdx.x;
    const int i0 = tile * (kThreads * V);

    // preamble: window starts of this tile, once per edge
    if (tid < dv) {
        const EdgeDesc d = tab.edge[cd.ebeg + tid];
        int r0 = i0 - d.shift; r0 += (r0 < 0) ? Z : 0;       // check index of the tile's first variable
        int qo = -1;
        if (d.p_off >= 0) { int x = i0 + d.delta; x -= (x >= Z) ? Z : 0; qo = d.p_off + x; }
        s_eo[tid] = make_int2(qo < 0 ? -1 : 4 * qo, 4 * (d.t_off + r0));    // byte offsets
    }
    if (tid < ng) s_gd[tid] = tab.gen[cd.gbeg + tid];
    if (EXACT) {
        if (tid < NG * PCAP) {                               // slot (g, jj): partner jj of gen edge g, or -1
            const int g = tid / PCAP, jj = tid - g * PCAP;
            const GenDesc gd = tab.gen[cd.gbeg + g];
            int po = -1;
            if (jj < gd.np) {
                const PartnerDesc p = tab.partner[cd.pbeg + gd.pbeg + jj];
                int x = i0 + p.delta; x -= (x >= Z) ? Z : 0;
                po = 4 * (p.off + x);
            }
            s_po[tid] = po;
        }
    } else {
#pragma unroll 1
        for (int j = tid; j < cd.np; j += kThreads) {
            const PartnerDesc p = tab.partner[cd.pbeg + j];
            int x = i0 + p.delta; x -= (x >= Z) ? Z : 0;
            s_po[j] = 4 * (p.off + x);
        }
    }
    __syncthreads();

    const float* __restrict__ qP = a.qb[in_buf] + (int64_t)f * a.EZs + tid;
    const float* __restrict__ tP = a.t + (int64_t)f * a.mZs + tid;
    float Q[V];
    bool valid[V];
    unsigned xb[V];
#pragma unroll
    for (int v = 0; v < V; ++v) {
        const int i = i0 + v * kThreads + tid;
        valid[v] = i < Z;
        Q[v] = valid[v] ? llr_to_log2(__ldg(a.llr + (int64_t)f * a.n + (int64_t)cd.col * Z + i)) : 0.0f;
        xb[v] = (!FINAL && ng > 0) ? a.hard_in[(int64_t)f * a.AZs + (int64_t)ca * Zs + i] : 0u;
    }

    // phase 1: all loads.  Gen partners first (EXACT: fixed slots, predicated off where the row is shorter)
    float pw[EXACT ? NGS : 1][EXACT ? PCAP : 1][V];
    if (EXACT) {
#pragma unroll
        for (int g = 0; g < NG; ++g) {
#pragma unroll
            for (int j = 0; j < PCAP; ++j) {
                const int po = s_po[g * PCAP + j];
#pragma unroll
                for (int v = 0; v < V; ++v)
                    pw[g][j][v] = (po != -1) ? __ldg(byte_ptr(qP, po) + v * kThreads) : 0.0f;
            }
        }
    }
    float tv[DV][V], wv[DV][V];
#pragma unroll UNR
    for (int k = 0; k < (EXACT ? DV : dv); ++k) {
        const int2 o = s_eo[k];
#pragma unroll
        for (int v = 0; v < V; ++v) tv[k][v] = __ldg(byte_ptr(tP, o.y) + v * kThreads);
        if (EXACT ? (k >= NG) : (o.x != -1)) {
#pragma unroll
            for (int v = 0; v < V; ++v) wv[k][v] = __ldg(byte_ptr(qP, o.x) + v * kThreads);
        }
    }

    // phase 2: gen rows: fold the partners into one equivalent q (the rule is associative); bit 0 of a gen edge's
    // state is its variable's hard decision, so the XOR of the raw words carries sign product AND parity
    unsigned bad = 0;
#pragma unroll UNG
    for (int g = 0; g < (EXACT ? NG : ng); ++g) {
        const GenDesc gd = s_gd[g];
        float num[V], den[V];
        unsigned xa[V];
#pragma unroll
        for (int v = 0; v < V; ++v) { num[v] = 0.0f; den[v] = 1.0f; xa[v] = 0u; }
        if (EXACT) {
            // an empty slot holds +0.0: the identity of both the XOR and the fold
#pragma unroll
            for (int j = 0; j < PCAP; ++j) {
#pragma unroll
                for (int v = 0; v < V; ++v) {
                    const unsigned wb = __float_as_uint(pw[EXACT ? g : 0][EXACT ? j : 0][v]);
                    xa[v] ^= wb;
                    boxplus_acc(__uint_as_float(wb & 0x7ffffffeu), num[v], den[v]);
                }
            }
#pragma unroll 1
            for (int j = PCAP; j < gd.np; ++j) {             // rows of degree > PCAP + 1: rare, slow path
                const PartnerDesc p = tab.partner[cd.pbeg + gd.pbeg + j];
                int x = i0 + p.delta; x -= (x >= Z) ? Z : 0;
#pragma unroll
                for (int v = 0; v < V; ++v) {
                    const unsigned wb = __float_as_uint(__ldg(qP + p.off + x + v * kThreads));
                    xa[v] ^= wb;
                    boxplus_acc(__uint_as_float(wb & 0x7ffffffeu), num[v], den[v]);
                }
            }
        } else {
#pragma unroll 4
            for (int j = 0; j < gd.np; ++j) {
                const int po = s_po[gd.pbeg + j];
#pragma unroll
                for (int v = 0; v < V; ++v) {
                    const unsigned wb = __float_as_uint(__ldg(byte_ptr(qP, po) + v * kThreads));
                    xa[v] ^= wb;
                    boxplus_acc(__uint_as_float(wb & 0x7ffffffeu), num[v], den[v]);
                }
            }
        }
#pragma unroll
        for (int v = 0; v < V; ++v) {
            wv[g][v] = with_sign(num[v] * rcp_approx(den[v]), xa[v] & 0x80000000u);
            if (!FINAL && gd.counter)    // parity of the row at the input iteration: s_c ^ XOR xhat (t = (-1)^{s_c} 0)
                bad |= (xa[v] ^ xb[v] ^ (__float_as_uint(tv[g][v]) >> 31)) & (valid[v] ? 1u : 0u);
        }
    }

    // phase 3: check-node rule: partner [+] static term; the sign product includes (-1)^{s_c} via t
#pragma unroll UNR
    for (int k = 0; k < (EXACT ? DV : dv); ++k) {
#pragma unroll
        for (int v = 0; v < V; ++v) {
            const float qa = fabsf(wv[k][v]), tt = fabsf(tv[k][v]);
            const float mag = mag_of(qa + tt, fmaf(qa, tt, 1.0f));
            tv[k][v] = with_sign(mag, sign_of(wv[k][v]) ^ sign_of(tv[k][v]));   // tv now holds m'_cv
        }
    }

    // phase 4: variable-node rule
    float suf[DV + 1][V];
#pragma unroll
    for (int v = 0; v < V; ++v) suf[EXACT ? DV : dv][v] = 0.0f;
#pragma unroll UNR
    for (int k = (EXACT ? DV : dv) - 1; k >= 0; --k) {
#pragma unroll
        for (int v = 0; v < V; ++v) suf[k][v] = suf[k + 1][v] + tv[k][v];
    }
    unsigned xh[V];
#pragma unroll
    for (int v = 0; v < V; ++v) {
        const float L = Q[v] + suf[0][v];                    // L'_v
        xh[v] = __float_as_uint(L) >> 31;                    // 0 iff L_v >= 0
        const int i = i0 + v * kThreads + tid;
        if (FINAL) {
            if (valid[v]) {
                const int64_t vv = (int64_t)f * a.n + (int64_t)cd.col * Z + i;
                a.d_hard[vv] = (uint8_t)xh[v];
                if (a.d_post) a.d_post[vv] = L * kLn2;
            }
        } else {
            a.hard_out[(int64_t)f * a.AZs + (int64_t)ca * Zs + i] = (uint8_t)xh[v];
        }
    }
    if (FINAL) return;

    if (ng > 0 && __any_sync(0xffffffffu, bad != 0) && (tid & 31) == 0) a.topbad[f] = 1;

    // tiles that own the first kHalo entries of the run write them twice (run + halo)
    const int nrep = (i0 < kHalo) ? 2 : 1;
#pragma unroll 1
    for (int rep = 0; rep < nrep; ++rep) {
        float* __restrict__ sp = a.qb[a.out_buf] + (int64_t)f * a.EZs + (int64_t)cd.ebeg * Zs + (rep ? Z : 0) + i0 + tid;
        float run[V];
#pragma unroll
        for (int v = 0; v < V; ++v) run[v] = Q[v];
#pragma unroll UNR
        for (int k = 0; k < (EXACT ? DV : dv); ++k) {
#pragma unroll
            for (int v = 0; v < V; ++v) {
                const float Lvc = run[v] + suf[k + 1][v];    // Q + sum_{k' != k} m_k'
                run[v] += tv[k][v];
                unsigned wb = __float_as_uint(w_of(Lvc));
                if (k < ng) wb = (wb & 0xfffffffeu) | xh[v]; // gen edge: tag with the hard decision
                if (valid[v]) sp[v * kThreads] = __uint_as_float(wb);
            }
            sp = byte_ptr(sp, 4u * Zs);
        }
    }
}

template <int DV, int NG, int PCAP, bool EXACT>
void launch_pass(const PassLaunch& L) {
    if (L.V == 2 && EXACT) {
        if (L.final_mode) k_pass<DV, NG, PCAP, EXACT, 2, true><<<L.grid, kThreads, 0, L.stream>>>(L.tab, L.args);
        else k_pass<DV, NG, PCAP, EXACT, 2, false><<<L.grid, kThreads, 0, L.stream>>>(L.tab, L.args);
    } else {
        if (L.final_mode) k_pass<DV, NG, PCAP, EXACT, 1, true><<<L.grid, kThreads, 0, L.stream>>>(L.tab, L.args);
        else k_pass<DV, NG, PCAP, EXACT, 1, false><<<L.grid, kThreads, 0, L.stream>>>(L.tab, L.args);
    }
}

}  // namespace qc

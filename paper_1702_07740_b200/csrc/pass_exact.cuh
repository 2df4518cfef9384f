// k_pass_exact -- the fused flooding iteration (steps a1 + a2 + the cheap part of a3, Algorithm 1 steps 2-4)
// for codes whose active columns all have the same shape: DV edges, the first NG of them into gen rows (the
// BASELINE.json codes: 11 or 21 edges, 3 into the top rows).  Same arithmetic as k_pass (pass_kernel.cuh); what differs
// is where the tables live: the column descriptors travel in the kernel PARAMETERS (constant bank), so the preamble that
// forms the block-uniform window starts (one thread per stream, into shared memory) reads no global memory: the first
// state load is issued a few hundred cycles after the CTA starts instead of after three dependent L2 round trips.
#pragma once

#include "check.cuh"
#include "common.cuh"

namespace qc {

template <int DV, int NG, int PCAP, int V, bool FINAL>
__global__ void __launch_bounds__(kThreads, V == 1 ? 7 : 4) k_pass_exact(const __grid_constant__ ExactTable<DV, NG, PCAP> T,
                                                         const __grid_constant__ PassArgs a,
                                                         const PartnerDesc* __restrict__ partner,
                                                         const CheckTables ctab, const __grid_constant__ CheckArgs chk) {
    constexpr int NGS = NG > 0 ? NG : 1;
    pdl_launch();
    if (!FINAL && (int)blockIdx.y == a.cand_y) {             // the extra grid row: early-exit check of iteration t-2
        pdl_wait();
        cand_work(ctab, chk, blockIdx.z * gridDim.x + blockIdx.x, gridDim.x * gridDim.z, threadIdx.x, kThreads);
        return;
    }
    const int f = a.flip ? gridDim.z - 1 - blockIdx.z : blockIdx.z;
    const int ca = blockIdx.y;                               // block-uniform active column
    const ExactCol<DV, NG, PCAP>& cd = T.c[ca];
    const int Z = a.Z, Zs = a.Zs;
    const int tid = threadIdx.x;
    const int i0 = blockIdx.x * (kThreads * V);

    // preamble: window starts of this tile as byte offsets, one thread per stream
    // byte offsets are formed in UNSIGNED arithmetic: a frame's runs stay below 2^30 floats (qcldpc_code_create)
    __shared__ uint2 s_eo[DV];
    __shared__ unsigned s_po[NGS * PCAP];
    static_assert(DV <= kThreads && NGS * PCAP <= kThreads, "one preamble thread per stream");
    if (tid < DV) {
        int r0 = i0 - cd.shift[tid]; r0 += (r0 < 0) ? Z : 0;  // check index of the tile's first variable
        int x = i0 + cd.delta[tid]; x -= (x >= Z) ? Z : 0;
        s_eo[tid] = make_uint2(4u * (unsigned)(cd.p_off[tid] + x), 4u * (unsigned)(cd.t_off[tid] + r0));
    }
    if (NG > 0 && tid >= kThreads - NG * PCAP) {             // slot (g, j): partner j of gen edge g, or -1
        const int sl = tid - (kThreads - NG * PCAP);
        int x = i0 + cd.g_delta[sl]; x -= (x >= Z) ? Z : 0;
        s_po[sl] = cd.g_off[sl] >= 0 ? 4u * (unsigned)(cd.g_off[sl] + x) : 0xffffffffu;   // no partner in this slot
    }
    pdl_wait();                                              // from here on: memory the previous launch wrote
    int in_buf;
    if (FINAL) {
        const int Tit = a.iters[f];
        if (Tit <= 0) return;                                // t = 0: k_init_cols wrote the outputs
        in_buf = (Tit + 3) % 4;                              // w^(T-1)
    } else {
        if (a.done[f]) return;                               // frame already stopped: its state stays frozen
        in_buf = a.in_buf;
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
        xb[v] = (!FINAL && NG > 0) ? a.hard_in[(int64_t)f * a.AZs + (int64_t)ca * Zs + i] : 0u;
    }

    // phase 1: every load, back to back.  Window starts are block-uniform (halo layout, common.cuh).
    float pw[NGS][PCAP][V];
#pragma unroll
    for (int g = 0; g < NG; ++g) {
#pragma unroll
        for (int j = 0; j < PCAP; ++j) {
            const unsigned po = s_po[g * PCAP + j];          // 0xffffffff: the row has fewer partners
#pragma unroll
            for (int v = 0; v < V; ++v)
                pw[g][j][v] = (po != 0xffffffffu) ? __ldg(byte_ptr(qP, po) + v * kThreads) : 0.0f;
        }
    }
    float tv[DV][V], wv[DV][V];
#pragma unroll
    for (int k = 0; k < DV; ++k) {
        const uint2 o = s_eo[k];
#pragma unroll
        for (int v = 0; v < V; ++v) tv[k][v] = __ldg(byte_ptr(tP, o.y) + v * kThreads);
        if (k >= NG) {
#pragma unroll
            for (int v = 0; v < V; ++v) wv[k][v] = __ldg(byte_ptr(qP, o.x) + v * kThreads);
        }
    }

    // phase 2: gen rows: fold the partners into one equivalent q (the rule is associative); bit 0 of a gen edge's
    // state is its variable's hard decision, so the XOR of the raw words carries sign product AND parity
    unsigned bad = 0;
#pragma unroll
    for (int g = 0; g < NG; ++g) {
        float num[V], den[V];
        unsigned xa[V];
#pragma unroll
        for (int v = 0; v < V; ++v) { num[v] = 0.0f; den[v] = 1.0f; xa[v] = 0u; }
        // an empty slot holds +0.0: the identity of both the XOR and the fold
#pragma unroll
        for (int j = 0; j < PCAP; ++j) {
#pragma unroll
            for (int v = 0; v < V; ++v) {
                const unsigned wb = __float_as_uint(pw[g][j][v]);
                xa[v] ^= wb;
                boxplus_acc(__uint_as_float(wb & 0x7ffffffeu), num[v], den[v]);
            }
        }
        const int np = cd.g_np[g];
#pragma unroll 1
        for (int j = PCAP; j < np; ++j) {                    // rows of degree > PCAP + 1: rare, slow path
            const PartnerDesc p = partner[cd.g_pbeg[g] + j];
            int x = i0 + p.delta; x -= (x >= Z) ? Z : 0;
#pragma unroll
            for (int v = 0; v < V; ++v) {
                const unsigned wb = __float_as_uint(__ldg(qP + p.off + x + v * kThreads));
                xa[v] ^= wb;
                boxplus_acc(__uint_as_float(wb & 0x7ffffffeu), num[v], den[v]);
            }
        }
#pragma unroll
        for (int v = 0; v < V; ++v) {
            wv[g][v] = with_sign(num[v] * rcp_approx(den[v]), xa[v] & 0x80000000u);
            if (!FINAL && cd.g_counter[g])   // parity of the row at the input iteration: s_c ^ XOR xhat (t = (-1)^{s_c} 0)
                bad |= (xa[v] ^ xb[v] ^ (__float_as_uint(tv[g][v]) >> 31)) & (valid[v] ? 1u : 0u);
        }
    }

    // phase 3: check-node rule: partner [+] static term; the sign product includes (-1)^{s_c} via t
#pragma unroll
    for (int k = 0; k < DV; ++k) {
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
    for (int v = 0; v < V; ++v) suf[DV][v] = 0.0f;
#pragma unroll
    for (int k = DV - 1; k >= 0; --k) {
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

    if (NG > 0 && __any_sync(0xffffffffu, bad != 0) && (tid & 31) == 0) a.topbad[f] = 1;

    // tiles that own the first kHalo entries of the run write them twice (run + halo)
    const int nrep = (i0 < kHalo) ? 2 : 1;
#pragma unroll 1
    for (int rep = 0; rep < nrep; ++rep) {
        float* __restrict__ sp = a.qb[a.out_buf] + (int64_t)f * a.EZs + (int64_t)cd.ebeg * Zs + (rep ? Z : 0) + i0 + tid;
        float run[V];
#pragma unroll
        for (int v = 0; v < V; ++v) run[v] = Q[v];
#pragma unroll
        for (int k = 0; k < DV; ++k) {
#pragma unroll
            for (int v = 0; v < V; ++v) {
                const float Lvc = run[v] + suf[k + 1][v];    // Q + sum_{k' != k} m_k'
                run[v] += tv[k][v];
                unsigned wb = __float_as_uint(w_of(Lvc));
                if (k < NG) wb = (wb & 0xfffffffeu) | xh[v]; // gen edge: tag with the hard decision
                if (valid[v]) sp[v * kThreads] = __uint_as_float(wb);
            }
            sp = byte_ptr(sp, 4u * Zs);
        }
    }
}

}  // namespace qc

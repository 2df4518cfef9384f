// k_pass -- steps a1 + a2 (+ the cheap part of a3) of the hot path: one flooding iteration of Algorithm 1 (steps 2-4,
// P:348-363), fused and VN-centric, for ANY code the handle accepts (active column degree <= kMaxDv, any row degree,
// any Z): the correctness path for general codes and the path of the paper's own ensemble (NEXT-1: ~800 active
// columns of degree 59/60 per 20,000, circulants of q = 21 or 50).  Codes whose columns all have one of
// the BASELINE.json shapes run k_pass_exact (pass_exact.cuh) instead.
//
// One CTA = TB consecutive variables of one active column of one frame (TB = 32, 64 or 128: the smallest that covers Z,
// so that circulants of 21 or 50 do not idle most of a 128-thread block).  Runs are stored compactly (no halo); a tile
// reads the cyclic window [x0, x0 + TB) of a run with one compare-subtract per element, x0 block-uniform from the
// preamble (tables in shared memory).
//   edges are processed in chunks of kChunk with all loads of a chunk in flight: t of the row, then either the single
//   partner (pair row: two active edges + one absorbed variable) or the fold of all other edges of a gen row; the
//   row's counter edge also forms the parity of the PREVIOUS iteration's hard decisions from the bit-0 tags;
//   check-node rule per edge -> m[k] (registers, compile-time indexed);
//   variable-node rule: L_v = Q_v + sum m, xhat_v, L_vc = L_v - m_cv (the LLR-domain difference is
//   benign: |m| <= 30; the cancellation hazard of SURVEY N3 is on the check-node side, where exclusion stays direct).
// FINAL = true: same arithmetic on each frame's frozen state, writes the outputs (hard bits, posterior) instead.
#pragma once

#include "common.cuh"

namespace qc {

constexpr int kChunk = 8;
constexpr int kGenSlots = 2;                                 // partners of a gen edge loaded with its chunk

struct StreamDesc { unsigned base, x0; };                     // element (x0 + lane) mod Z of the run at float index base

template <int TB>
struct PassCtx {
    const float* qP; const float* tP;                        // this frame's edge state (input buffer) and static terms
    const StreamDesc* s_t; const StreamDesc* s_p; const GenDesc* s_gd; const StreamDesc* s_po;
    float* s_m;                                              // messages of this thread: s_m[k * TB]
    unsigned lane, Z, xb;
    int dv, ng;
    bool valid;
    float sum; unsigned bad;
};

#ifdef __CUDACC__
// unsigned index arithmetic and one 32x32+64 multiply-add per address (runs start below 2^30 floats: code_create)
__device__ __forceinline__ float load_stream(const float* p, const StreamDesc sd, unsigned lane, unsigned Z) {
    unsigned idx = sd.x0 + lane;
    idx -= (idx >= Z) ? Z : 0u;
    return __ldg(byte_ptr(p, 4u * (sd.base + idx)));
}

// check-node rule: partner [+] static term; the sign product includes (-1)^{s_c} via t
__device__ __forceinline__ float cn_rule(float wv, float tv) {
    const float qa = fabsf(wv), tt = fabsf(tv);
    return with_sign(mag_of(qa + tt, fmaf(qa, tt, 1.0f)), sign_of(wv) ^ sign_of(tv));
}

// One chunk of kChunk edges starting at edge k0: loads back to back, then the check-node rule, messages to shared memory.
// MODE 1: all edges are pair edges (k0 >= ng, k0 + kChunk <= dv); MODE 2: all are gen edges (k0 + kChunk <= ng); MODE 0:
// anything (per-edge predicates).
template <int TB, bool FINAL, int MODE>
__device__ __forceinline__ void chunk_cn(PassCtx<TB>& cx, const int k0) {
    float tv[kChunk], wv[kChunk];
    if (MODE == 1) {
#pragma unroll
        for (int j = 0; j < kChunk; ++j) {
            tv[j] = load_stream(cx.tP, cx.s_t[k0 + j], cx.lane, cx.Z);
            wv[j] = load_stream(cx.qP, cx.s_p[k0 + j], cx.lane, cx.Z);
        }
#pragma unroll
        for (int j = 0; j < kChunk; ++j) {
            const float mk = cn_rule(wv[j], tv[j]);
            cx.s_m[(k0 + j) * TB] = mk;
            cx.sum += mk;
        }
        return;
    }
    float pw[kChunk][kGenSlots];
    int np[kChunk], pbeg[kChunk], ctr[kChunk];
#pragma unroll
    for (int j = 0; j < kChunk; ++j) {                       // loads of the chunk, back to back
        const int k = k0 + j;
        tv[j] = 0.0f; wv[j] = 0.0f; np[j] = 0; pbeg[j] = 0; ctr[j] = 0;
#pragma unroll
        for (int jj = 0; jj < kGenSlots; ++jj) pw[j][jj] = 0.0f;
        if (MODE == 2 || k < cx.dv) {
            tv[j] = load_stream(cx.tP, cx.s_t[k], cx.lane, cx.Z);
            if (MODE == 2 || k < cx.ng) {                    // gen edge: its first kGenSlots partners travel with the
                const GenDesc gd = cx.s_gd[k];               // chunk's other loads (empty slot: +0.0, the identity)
                np[j] = gd.np; pbeg[j] = gd.pbeg; ctr[j] = gd.counter;
#pragma unroll
                for (int jj = 0; jj < kGenSlots; ++jj)
                    if (jj < gd.np) pw[j][jj] = load_stream(cx.qP, cx.s_po[gd.pbeg + jj], cx.lane, cx.Z);
            } else {
                wv[j] = load_stream(cx.qP, cx.s_p[k], cx.lane, cx.Z);
            }
        }
    }
#pragma unroll
    for (int j = 0; j < kChunk; ++j) {
        const int k = k0 + j;
        if (MODE == 2 || k < cx.ng) {
            // gen row: fold the other edges into one equivalent q (the rule is associative); bit 0 of a gen edge's
            // state is its variable's hard decision: the XOR of the raw words carries sign AND parity
            float num = 0.0f, den = 1.0f;
            unsigned xa = 0u;
#pragma unroll
            for (int jj = 0; jj < kGenSlots; ++jj) {
                const unsigned wb = __float_as_uint(pw[j][jj]);
                xa ^= wb;
                boxplus_acc(__uint_as_float(wb & 0x7ffffffeu), num, den);
            }
#pragma unroll 1
            for (int jj = kGenSlots; jj < np[j]; ++jj) {     // rows of degree > kGenSlots + 1
                const unsigned wb = __float_as_uint(load_stream(cx.qP, cx.s_po[pbeg[j] + jj], cx.lane, cx.Z));
                xa ^= wb;
                boxplus_acc(__uint_as_float(wb & 0x7ffffffeu), num, den);
            }
            wv[j] = with_sign(num * rcp_approx(den), xa & 0x80000000u);
            if (!FINAL && ctr[j])            // parity of the row at the input iteration (t = (-1)^{s_c} 0 there)
                cx.bad |= (xa ^ cx.xb ^ (__float_as_uint(tv[j]) >> 31)) & (cx.valid ? 1u : 0u);
        }
        if (MODE == 2 || k < cx.dv) {
            const float mk = cn_rule(wv[j], tv[j]);
            cx.s_m[k * TB] = mk;
            cx.sum += mk;
        }
    }
}
#endif

// dynamic shared memory: stream tables, then the messages m'_cv of the tile, [max_dv][TB] floats
inline size_t pass_any_table_bytes(int max_np) {
    return (size_t)kMaxDv * (2 * sizeof(StreamDesc) + sizeof(GenDesc)) + (size_t)(max_np > 0 ? max_np : 1) * sizeof(StreamDesc);
}
inline size_t pass_any_smem(int max_np, int max_dv, int tb, int groups) {
    return pass_any_table_bytes(max_np) + (size_t)((max_dv > 0 ? max_dv : 1) + groups) * tb * sizeof(float);
}

// G = edge groups: the CTA is TB x G threads, thread (tid, grp) handles the chunks grp, grp + G, ... of the column's
// edges, so a column of degree 60 is four chains of 15 edges instead of one of 60 (the pass of a single frame is bound
// by that chain's latency); the partial sums of the groups meet in shared memory.
template <int TB, int G, bool FINAL>
__global__ void __launch_bounds__(TB * G, 1024 / (TB * G)) k_pass(const PassTables tab, const PassArgs a) {
    extern __shared__ __align__(16) unsigned char smem_any[];
    StreamDesc* const s_t = reinterpret_cast<StreamDesc*>(smem_any);          // [kMaxDv] t of edge k
    StreamDesc* const s_p = s_t + kMaxDv;                                     // [kMaxDv] partner of pair edge k
    GenDesc* const s_gd = reinterpret_cast<GenDesc*>(s_p + kMaxDv);           // [kMaxDv] gen edges
    StreamDesc* const s_po = reinterpret_cast<StreamDesc*>(s_gd + kMaxDv);    // [np] partners of the gen edges
    float* const s_m = reinterpret_cast<float*>(smem_any + a.table_bytes) + threadIdx.x;   // m'_cv of edge k: s_m[k * TB]
    float* const s_part = reinterpret_cast<float*>(smem_any + a.table_bytes) + a.max_dv * TB;   // [G][TB] partial sums

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
    const int tid = threadIdx.x, grp = threadIdx.y;
    const int flat = grp * TB + tid;
    const int i0 = tile * TB;
    const int i = i0 + tid;
    const bool valid = i < Z;
    const int lane = valid ? tid : 0;                        // idle threads read element 0 of every window

    // preamble: window starts of this tile, once per stream
    for (int k = flat; k < dv; k += TB * G) {
        const EdgeDesc d = tab.edge[cd.ebeg + k];
        int r0 = (i0 - d.shift) % Z; r0 += (r0 < 0) ? Z : 0;  // check index of the tile's first variable
        s_t[k] = StreamDesc{(unsigned)d.t_off, (unsigned)r0};
        s_p[k] = StreamDesc{(unsigned)(d.p_off >= 0 ? d.p_off : 0), (unsigned)(d.p_off >= 0 ? (i0 + d.delta) % Z : 0)};
    }
    for (int g = flat; g < ng; g += TB * G) s_gd[g] = tab.gen[cd.gbeg + g];
    for (int j = flat; j < cd.np; j += TB * G) {
        const PartnerDesc p = tab.partner[cd.pbeg + j];
        s_po[j] = StreamDesc{(unsigned)p.off, (unsigned)((i0 + p.delta) % Z)};
    }
    __syncthreads();

    // opaque to the optimiser: otherwise the two frame pointers are re-formed (64-bit multiply, constant loads) at
    // every one of the ~150 loads of a thread
    unsigned long long qP_u = reinterpret_cast<unsigned long long>(a.qb[in_buf] + (int64_t)f * a.EZs);
    unsigned long long tP_u = reinterpret_cast<unsigned long long>(a.t + (int64_t)f * a.mZs);
    asm volatile("" : "+l"(qP_u), "+l"(tP_u));
    PassCtx<TB> cx;
    cx.qP = reinterpret_cast<const float*>(qP_u); cx.tP = reinterpret_cast<const float*>(tP_u);
    cx.s_t = s_t; cx.s_p = s_p; cx.s_gd = s_gd; cx.s_po = s_po; cx.s_m = s_m;
    cx.lane = (unsigned)lane; cx.Z = (unsigned)Z; cx.dv = dv; cx.ng = ng;
    cx.xb = (!FINAL && ng > 0) ? a.hard_in[(int64_t)f * a.AZs + (int64_t)ca * Zs + (valid ? i : 0)] : 0u;
    cx.valid = valid; cx.sum = 0.0f; cx.bad = 0u;
    const float Q = valid ? llr_to_log2(__ldg(a.llr + (int64_t)f * a.n + (int64_t)cd.col * Z + i)) : 0.0f;

    // The chunk loop is NOT unrolled (a fully unrolled body for 64 edges is 170 KB of code: the pass becomes bound by
    // instruction fetch); the messages of the tile wait in shared memory for the variable-node rule instead.  A chunk
    // whose 8 edges are all pair edges, or all gen edges, runs a body without per-edge predicates.
#pragma unroll 1
    for (int k0 = grp * kChunk; k0 < dv; k0 += G * kChunk) {
        if (k0 >= ng && k0 + kChunk <= dv) chunk_cn<TB, FINAL, 1>(cx, k0);
        else if (k0 + kChunk <= ng) chunk_cn<TB, FINAL, 2>(cx, k0);
        else chunk_cn<TB, FINAL, 0>(cx, k0);
    }
    float sum = cx.sum;

    // variable-node rule
    if (G > 1) {                                             // the groups' partial sums meet here, in a fixed order
        s_part[grp * TB + tid] = sum;
        __syncthreads();
        sum = 0.0f;
#pragma unroll
        for (int g = 0; g < G; ++g) sum += s_part[g * TB + tid];
    }
    const float L = Q + sum;                                 // L'_v
    const unsigned xh = __float_as_uint(L) >> 31;            // 0 iff L_v >= 0
    if (FINAL) {
        if (valid && grp == 0) {
            const int64_t vv = (int64_t)f * a.n + (int64_t)cd.col * Z + i;
            a.d_hard[vv] = (uint8_t)xh;
            if (a.d_post) a.d_post[vv] = L * kLn2;
        }
        return;
    }
    if (valid && grp == 0) a.hard_out[(int64_t)f * a.AZs + (int64_t)ca * Zs + i] = (uint8_t)xh;
    if (ng > 0 && __any_sync(0xffffffffu, cx.bad != 0) && (tid & 31) == 0) a.topbad[f] = 1;

    float* const sp = a.qb[a.out_buf] + (int64_t)f * a.EZs + (int64_t)cd.ebeg * Zs + (valid ? i : 0);
    const unsigned Zs4 = 4u * (unsigned)Zs;
    const bool single = dv == 1;                             // a single edge sends Q itself
#pragma unroll 1
    for (int k0 = grp * kChunk; k0 < dv; k0 += G * kChunk) {
        if (k0 >= ng && k0 + kChunk <= dv) {                 // eight pair edges: no tags, no bounds
#pragma unroll
            for (int j = 0; j < kChunk; ++j) {
                const float Lvc = single ? Q : L - s_m[(k0 + j) * TB];   // Q + sum_{k' != k} m_k'
                if (valid) *byte_ptr(sp, (unsigned)(k0 + j) * Zs4) = w_of(Lvc);
            }
        } else {
#pragma unroll
            for (int j = 0; j < kChunk; ++j) {
                const int k = k0 + j;
                if (k < dv) {
                    const float Lvc = single ? Q : L - s_m[k * TB];
                    unsigned wb = __float_as_uint(w_of(Lvc));
                    if (k < ng) wb = (wb & 0xfffffffeu) | xh;    // gen edge: tag with the hard decision
                    if (valid) *byte_ptr(sp, (unsigned)k * Zs4) = __uint_as_float(wb);
                }
            }
        }
    }
}

template <int TB, int G>
inline void launch_pass_tb(const PassLaunch& L, PassArgs args) {
    args.tiles = (args.Z + TB - 1) / TB;
    args.max_dv = L.max_dv > 0 ? L.max_dv : 1;
    const size_t smem = pass_any_smem(L.max_np, L.max_dv, TB, G);
    static thread_local bool attr_set = false;
    if (!attr_set) {            // tables (<= 18.4 KB) + messages (<= 32 KB) can exceed the 48 KB default
        cudaFuncSetAttribute(k_pass<TB, G, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
        cudaFuncSetAttribute(k_pass<TB, G, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
        attr_set = true;
    }
    const dim3 grid(args.tiles * L.n_cols, L.n_frames), block(TB, G);
    if (L.final_mode) k_pass<TB, G, true><<<grid, block, smem, L.stream>>>(L.tab, args);
    else launch_pdl(k_pass<TB, G, false>, grid, block, smem, L.stream, L.tab, args);
}

inline void launch_pass_any(const PassLaunch& L) {
    PassArgs args = L.args;
    args.table_bytes = (int)pass_any_table_bytes(L.max_np);
    const int Z = args.Z;
    const bool split = L.max_dv > 2 * kChunk;               // long columns: four edge groups per variable
    if (Z <= 32) { if (split) launch_pass_tb<32, 4>(L, args); else launch_pass_tb<32, 1>(L, args); }
    else if (Z <= 64) { if (split) launch_pass_tb<64, 4>(L, args); else launch_pass_tb<64, 1>(L, args); }
    else { if (split) launch_pass_tb<128, 4>(L, args); else launch_pass_tb<128, 1>(L, args); }
}

}  // namespace qc

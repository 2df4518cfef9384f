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
//   partner (pair row: two active edges + one absorbed variable), the two partners of a triple row (three active
//   edges + one absorbed variable), or the fold of all other edges of a gen row; the row's counter edge also forms
//   the parity of the PREVIOUS iteration's hard decisions from the bit-0 tags;
//   check-node rule per edge -> m[k] (shared memory, one column of the tile per thread);
//   variable-node rule: L_v = Q_v + sum m, xhat_v, L_vc = L_v - m_cv (the LLR-domain difference is
//   benign: |m| <= 30; the cancellation hazard of SURVEY N3 is on the check-node side, where exclusion stays direct).
// FV = 2 (batched decodes): a thread carries the same variable of TWO frames; the table lookups, window indices and
// predicates -- most of this kernel's instructions -- are shared by the pair.
// PACK = true (batches of a code whose circulant is at most half a tile): a.pack frames side by side in the tile, thread
// tid = variable tid mod Z of frame tid / Z; liveness and frame pointers are then per lane.
// FINAL = true: same arithmetic on each frame's frozen state, writes the outputs (hard bits, posterior) instead.
#pragma once

#include "check.cuh"
#include "common.cuh"

#include <algorithm>

namespace qc {

constexpr int kChunk = 8;
constexpr int kGenSlots = 2;                                 // partners of a gen edge loaded with its chunk
constexpr int kGenMore = 4;                                  // further partners of a gen edge per round trip

struct StreamDesc { unsigned base, x0; };                     // element (x0 + lane) mod Z of the run at float index base

template <int TB, int FV>
struct PassCtx {
    const float* qP[FV]; const float* tP[FV];                // per frame: edge state (input buffer) and static terms
    const StreamDesc* s_t; const StreamDesc* s_p; const StreamDesc* s_p2; const GenDesc* s_gd; const StreamDesc* s_po;
    float* s_m;                                              // messages of this thread: s_m[(k * FV + v) * TB]
    unsigned lane, Z, xb[FV];
    int dv, ng;
    bool valid;
    float sum[FV]; unsigned bad[FV];
};

#ifdef __CUDACC__
// byte offset of this thread's element of a stream: unsigned arithmetic, runs start below 2^30 floats (code_create)
__device__ __forceinline__ unsigned stream_off(const StreamDesc sd, unsigned lane, unsigned Z) {
    const unsigned idx = sd.x0 + lane;                       // < 2 Z
    return 4u * (sd.base + min(idx, idx - Z));               // idx - Z wraps to a huge value when idx < Z
}

// One chunk of CH edges starting at edge k0: loads back to back, then the check-node rule, messages to shared memory.
// MODE 1: all edges are pair edges (k0 >= ng, k0 + CH <= dv); MODE 3: all are edges of triple rows (k0 >= ngh,
// k0 + CH <= ng); MODE 2: all are gen edges (k0 + CH <= ng); MODE 0: anything (per-edge predicates).
template <int TB, int FV, int CH, bool FINAL, int MODE>
__device__ __forceinline__ void chunk_cn(PassCtx<TB, FV>& cx, const int k0) {
    float tv[CH][FV], wv[CH][FV];
    if constexpr (MODE == 1) {
#pragma unroll
        for (int j = 0; j < CH; ++j) {
            const unsigned ot = stream_off(cx.s_t[k0 + j], cx.lane, cx.Z);
            const unsigned op = stream_off(cx.s_p[k0 + j], cx.lane, cx.Z);
#pragma unroll
            for (int v = 0; v < FV; ++v) {
                tv[j][v] = __ldg(byte_ptr(cx.tP[v], ot));
                wv[j][v] = __ldg(byte_ptr(cx.qP[v], op));
            }
        }
#pragma unroll
        for (int j = 0; j < CH; ++j) {
#pragma unroll
            for (int v = 0; v < FV; ++v) {
                const float mk = cn_rule(wv[j][v], tv[j][v]);
                cx.s_m[((k0 + j) * FV + v) * TB] = mk;
                cx.sum[v] += mk;
            }
        }
    } else if constexpr (MODE == 3) {
        // triple row: two partners, an absorbed variable, no parity to report.  (a [+] b) [+] |t| as one fraction:
        // num = a + b + |t| (1 + a b), den = 1 + a b + |t| (a + b): no reciprocal in between
        float pa[CH][FV], pb[CH][FV];
#pragma unroll
        for (int j = 0; j < CH; ++j) {
            const unsigned ot = stream_off(cx.s_t[k0 + j], cx.lane, cx.Z);
            const unsigned oa = stream_off(cx.s_p[k0 + j], cx.lane, cx.Z);
            const unsigned ob = stream_off(cx.s_p2[k0 + j], cx.lane, cx.Z);
#pragma unroll
            for (int v = 0; v < FV; ++v) {
                tv[j][v] = __ldg(byte_ptr(cx.tP[v], ot));
                pa[j][v] = __ldg(byte_ptr(cx.qP[v], oa));
                pb[j][v] = __ldg(byte_ptr(cx.qP[v], ob));
            }
        }
#pragma unroll
        for (int j = 0; j < CH; ++j) {
#pragma unroll
            for (int v = 0; v < FV; ++v) {
                const unsigned ua = __float_as_uint(pa[j][v]), ub = __float_as_uint(pb[j][v]);
                const float qa = __uint_as_float(ua & 0x7ffffffeu), qb = __uint_as_float(ub & 0x7ffffffeu);   // bit 0: tag
                float num = qa + qb, den = fmaf(qa, qb, 1.0f);
                boxplus_acc(fabsf(tv[j][v]), num, den);
                const float mk = with_sign(mag_of(num, den), (ua ^ ub ^ __float_as_uint(tv[j][v])) & 0x80000000u);
                cx.s_m[((k0 + j) * FV + v) * TB] = mk;
                cx.sum[v] += mk;
            }
        }
    } else {
    float pw[CH][kGenSlots][FV];
    int np[CH], pbeg[CH], ctr[CH];
#pragma unroll
    for (int j = 0; j < CH; ++j) {                           // loads of the chunk, back to back
        const int k = k0 + j;
        np[j] = 0; pbeg[j] = 0; ctr[j] = 0;
#pragma unroll
        for (int v = 0; v < FV; ++v) {
            tv[j][v] = 0.0f; wv[j][v] = 0.0f;
#pragma unroll
            for (int jj = 0; jj < kGenSlots; ++jj) pw[j][jj][v] = 0.0f;
        }
        if (MODE == 2 || k < cx.dv) {
            const unsigned ot = stream_off(cx.s_t[k], cx.lane, cx.Z);
#pragma unroll
            for (int v = 0; v < FV; ++v) tv[j][v] = __ldg(byte_ptr(cx.tP[v], ot));
            if (MODE == 2 || k < cx.ng) {                    // gen edge: its first kGenSlots partners travel with the
                const GenDesc gd = cx.s_gd[k];               // chunk's other loads (empty slot: +0.0, the identity)
                np[j] = gd.np; pbeg[j] = gd.pbeg; ctr[j] = gd.counter;
#pragma unroll
                for (int jj = 0; jj < kGenSlots; ++jj)
                    if (jj < gd.np) {
                        const unsigned op = stream_off(cx.s_po[gd.pbeg + jj], cx.lane, cx.Z);
#pragma unroll
                        for (int v = 0; v < FV; ++v) pw[j][jj][v] = __ldg(byte_ptr(cx.qP[v], op));
                    }
            } else {
                const unsigned op = stream_off(cx.s_p[k], cx.lane, cx.Z);
#pragma unroll
                for (int v = 0; v < FV; ++v) wv[j][v] = __ldg(byte_ptr(cx.qP[v], op));
            }
        }
    }
#pragma unroll
    for (int j = 0; j < CH; ++j) {
        const int k = k0 + j;
        if (MODE == 2 || k < cx.ng) {
            // gen row: fold the other edges into one equivalent q (the rule is associative); bit 0 of a gen edge's
            // state is its variable's hard decision: the XOR of the raw words carries sign AND parity
            float num[FV], den[FV];
            unsigned xa[FV];
#pragma unroll
            for (int v = 0; v < FV; ++v) {
                num[v] = 0.0f; den[v] = 1.0f; xa[v] = 0u;
#pragma unroll
                for (int jj = 0; jj < kGenSlots; ++jj) {
                    const unsigned wb = __float_as_uint(pw[j][jj][v]);
                    xa[v] ^= wb;
                    boxplus_acc(__uint_as_float(wb & 0x7ffffffeu), num[v], den[v]);
                }
            }
            // rows of degree > kGenSlots + 1: kGenMore partners per round trip (an empty slot is +0.0, the identity)
#pragma unroll 1
            for (int jb = kGenSlots; jb < np[j]; jb += kGenMore) {
                float pm[kGenMore][FV];
#pragma unroll
                for (int u = 0; u < kGenMore; ++u) {
                    const bool have = jb + u < np[j];
                    const unsigned op = stream_off(cx.s_po[pbeg[j] + (have ? jb + u : 0)], cx.lane, cx.Z);
#pragma unroll
                    for (int v = 0; v < FV; ++v) pm[u][v] = have ? __ldg(byte_ptr(cx.qP[v], op)) : 0.0f;
                }
#pragma unroll
                for (int u = 0; u < kGenMore; ++u)
#pragma unroll
                    for (int v = 0; v < FV; ++v) {
                        const unsigned wb = __float_as_uint(pm[u][v]);
                        xa[v] ^= wb;
                        boxplus_acc(__uint_as_float(wb & 0x7ffffffeu), num[v], den[v]);
                    }
            }
#pragma unroll
            for (int v = 0; v < FV; ++v) {
                if (!FINAL && ctr[j])        // parity of the row at the input iteration (t = (-1)^{s_c} 0 there)
                    cx.bad[v] |= (xa[v] ^ cx.xb[v] ^ (__float_as_uint(tv[j][v]) >> 31)) & (cx.valid ? 1u : 0u);
                // the static term joins the same fraction (as in MODE 3: an edge's message does not depend on the
                // body that computes it)
                boxplus_acc(fabsf(tv[j][v]), num[v], den[v]);
                const float mk = with_sign(mag_of(num[v], den[v]), (xa[v] ^ __float_as_uint(tv[j][v])) & 0x80000000u);
                cx.s_m[(k * FV + v) * TB] = mk;
                cx.sum[v] += mk;
            }
        } else if (k < cx.dv) {
#pragma unroll
            for (int v = 0; v < FV; ++v) {
                const float mk = cn_rule(wv[j][v], tv[j][v]);
                cx.s_m[(k * FV + v) * TB] = mk;
                cx.sum[v] += mk;
            }
        }
    }
    }   // MODE != 1
}
#endif

// dynamic shared memory: stream tables, then the messages m'_cv of the tile [max_dv][FV][TB], then partial sums [G][FV][TB]
inline size_t pass_any_table_bytes(int max_np) {
    return (size_t)kMaxDv * (3 * sizeof(StreamDesc) + sizeof(GenDesc)) + (size_t)(max_np > 0 ? max_np : 1) * sizeof(StreamDesc);
}
inline size_t pass_any_smem(int max_np, int max_dv, int tb, int groups, int fv) {
    return pass_any_table_bytes(max_np) + (size_t)((max_dv > 0 ? max_dv : 1) + groups) * fv * tb * sizeof(float);
}

// G = edge groups: the CTA is TB x G threads, thread (tid, grp) handles the chunks grp, grp + G, ... of the column's
// edges, so a column of degree 60 is four chains of 15 edges instead of one of 60 (the pass of a single frame is bound
// by that chain's latency); the partial sums of the groups meet in shared memory.
template <int TB, int G, int FV, bool FINAL, bool PACK>
__global__ void __launch_bounds__(TB * G, 1024 / (TB * G)) k_pass(const PassTables tab, const PassArgs a,
                                                                  const CheckTables ctab, const CheckArgs chk) {
    constexpr int CH = kChunk / FV;                           // edges per chunk: the loads in flight stay the same
    if (!FINAL && a.cand_y >= 0 && (int)blockIdx.x >= a.cand_y) {   // extra CTAs: early-exit check of iteration t-2
        pdl_launch();
        pdl_wait();
        cand_work(ctab, chk, blockIdx.y * (gridDim.x - a.cand_y) + (blockIdx.x - a.cand_y),
                  (gridDim.x - a.cand_y) * gridDim.y, threadIdx.y * TB + threadIdx.x, TB * G);
        return;
    }
    extern __shared__ __align__(16) unsigned char smem_any[];
    StreamDesc* const s_t = reinterpret_cast<StreamDesc*>(smem_any);          // [kMaxDv] t of edge k
    StreamDesc* const s_p = s_t + kMaxDv;                                     // [kMaxDv] partner of pair edge k
    StreamDesc* const s_p2 = s_p + kMaxDv;                                    // [kMaxDv] second partner of triple edge k
    GenDesc* const s_gd = reinterpret_cast<GenDesc*>(s_p2 + kMaxDv);          // [kMaxDv] gen edges
    StreamDesc* const s_po = reinterpret_cast<StreamDesc*>(s_gd + kMaxDv);    // [np] partners of the gen edges
    float* const s_m = reinterpret_cast<float*>(smem_any + a.table_bytes) + threadIdx.x;
    float* const s_part = reinterpret_cast<float*>(smem_any + a.table_bytes) + a.max_dv * FV * TB;

    // The loads of the prologue are ordered by dependence, not by meaning: the stop flags, the column descriptor and
    // then everything that hangs on it (edge tables, Q, last iteration's hard decisions) are in flight together, and
    // the flags are looked at last: three memory round trips before the first chunk instead of five.
    pdl_launch();
    const int ca = blockIdx.x / a.tiles;                     // block-uniform active column
    const int tile = blockIdx.x - ca * a.tiles;
    const ColDesc cd = tab.col[ca];                          // tables: constant, not the previous launch's output
    pdl_wait();
    // PACK: frames side by side in the tile when the circulant is at most half of it (one tile per column): thread
    // tid carries variable tid mod Z of the tile's frame tid / Z, so a circulant of 21 fills 63 of 64 lanes instead
    // of 21 of 32.  Frame of (CTA row y, v, sub) = (y FV + v) pack + sub; liveness is then per lane.
    const int Z = a.Z, Zs = a.Zs;
    const int tid = threadIdx.x, grp = threadIdx.y;
    const int sub_raw = PACK ? tid / Z : 0;
    const int i0 = tile * TB;
    const int li = tid - sub_raw * Z;                        // position in the tile's window
    const int i = i0 + li;
    const bool valid = PACK ? sub_raw < a.pack : i < Z;
    const int lane = valid ? li : 0;                         // idle threads read element 0 of every window
    const int row = a.flip ? (int)gridDim.y - 1 - (int)blockIdx.y : (int)blockIdx.y;   // CTA row of frames
    int fr[FV], in_buf[FV], flag[FV];
    bool live[FV];
#pragma unroll
    for (int v = 0; v < FV; ++v) {
        fr[v] = PACK ? (row * FV + v) * a.pack + (valid ? sub_raw : 0) : row * FV + v;
        live[v] = fr[v] < a.n_frames;
        fr[v] = live[v] ? fr[v] : a.n_frames - 1;            // out of range: any valid frame, nothing of it is stored
        if (PACK) live[v] = live[v] && valid;
        flag[v] = FINAL ? a.iters[fr[v]] : a.done[fr[v]];
    }
    const int dv = cd.dv, ng = cd.ng, ngh = cd.ngh;
    const int flat = grp * TB + tid;

    // window starts of this tile, once per stream
    for (int k = flat; k < dv; k += TB * G) {
        const EdgeDesc d = tab.edge[cd.ebeg + k];
        int r0 = i0 - d.shift; r0 += (r0 < 0) ? Z : 0;        // check index of the tile's first variable (i0, shift < Z)
        int x0 = i0 + d.delta; x0 -= (x0 >= Z) ? Z : 0;       // delta < Z: one wrap at most, no division
        int x1 = i0 + d.delta2; x1 -= (x1 >= Z) ? Z : 0;
        s_t[k] = StreamDesc{(unsigned)d.t_off, (unsigned)r0};
        s_p[k] = StreamDesc{(unsigned)(d.p_off >= 0 ? d.p_off : 0), (unsigned)(d.p_off >= 0 ? x0 : 0)};
        s_p2[k] = StreamDesc{(unsigned)(d.p2_off >= 0 ? d.p2_off : 0), (unsigned)(d.p2_off >= 0 ? x1 : 0)};
    }
    for (int g = flat; g < ng; g += TB * G) s_gd[g] = tab.gen[cd.gbeg + g];
    for (int j = flat; j < cd.np; j += TB * G) {
        const PartnerDesc p = tab.partner[cd.pbeg + j];
        int x0 = i0 + p.delta; x0 -= (x0 >= Z) ? Z : 0;
        s_po[j] = StreamDesc{(unsigned)p.off, (unsigned)x0};
    }
    PassCtx<TB, FV> cx;
    float Q[FV];
#pragma unroll
    for (int v = 0; v < FV; ++v) {
        cx.xb[v] = (!FINAL && ng > 0) ? a.hard_in[(int64_t)fr[v] * a.AZs + (int64_t)ca * Zs + (valid ? i : 0)] : 0u;
        Q[v] = valid ? llr_to_log2(__ldg(a.llr + (int64_t)fr[v] * a.n + (int64_t)cd.col * Z + i)) : 0.0f;
    }

    // a frame that is out of range or stopped is not live: it is computed on valid memory (the first live frame's
    // state; PACK: the frame's own, stale buffers) and nothing of it is stored; a CTA without a live frame leaves
    int f_any = -1;
#pragma unroll
    for (int v = 0; v < FV; ++v) {
        in_buf[v] = a.in_buf;
        if (FINAL) {
            live[v] = live[v] && flag[v] > 0;                // t = 0: k_init_cols wrote the outputs
            in_buf[v] = (flag[v] + 3) % 4;                   // w^(T-1): buffer (T - 1) mod 4
        } else {
            live[v] = live[v] && !flag[v];                   // frame already stopped: its state stays frozen
        }
        if (live[v] && f_any < 0) f_any = v;
    }
    if constexpr (PACK) {
        if (!__syncthreads_or(f_any >= 0)) return;           // the vote is also the barrier of the prologue
    } else {
        if (f_any < 0) return;
#pragma unroll
        for (int v = 0; v < FV; ++v)
            if (!live[v]) { fr[v] = fr[f_any]; in_buf[v] = in_buf[f_any]; }
        __syncthreads();
    }

#pragma unroll
    for (int v = 0; v < FV; ++v) {
        // opaque to the optimiser: otherwise the frame pointers are re-formed (64-bit multiply, constant loads) at
        // every one of the ~150 loads of a thread
        unsigned long long qP_u = reinterpret_cast<unsigned long long>(a.qb[in_buf[v]] + (int64_t)fr[v] * a.EZs);
        unsigned long long tP_u = reinterpret_cast<unsigned long long>(a.t + (int64_t)fr[v] * a.mZs);
        asm volatile("" : "+l"(qP_u), "+l"(tP_u));
        cx.qP[v] = reinterpret_cast<const float*>(qP_u);
        cx.tP[v] = reinterpret_cast<const float*>(tP_u);
        cx.sum[v] = 0.0f; cx.bad[v] = 0u;
    }
    cx.s_t = s_t; cx.s_p = s_p; cx.s_p2 = s_p2; cx.s_gd = s_gd; cx.s_po = s_po; cx.s_m = s_m;
    cx.lane = (unsigned)lane; cx.Z = (unsigned)Z; cx.dv = dv; cx.ng = ng; cx.valid = valid;

    // The chunk loop is NOT unrolled (a fully unrolled body for 64 edges is 170 KB of code: the pass becomes bound by
    // instruction fetch); the messages of the tile wait in shared memory for the variable-node rule instead.  A chunk
    // whose edges are all pair edges, all edges of triple rows, or all gen edges, runs a body without per-edge predicates.
    // Blocks of kChunk edges go to the groups in boustrophedon order (0 .. G-1, G-1 .. 0, ...: the group with the
    // column's first block, where the long gen rows are, gets the last, short one) whatever FV is, and every group
    // adds its messages in increasing k: a frame's result does not depend on the batch it is decoded in (bit for bit).
#pragma unroll 1
    for (int rnd = 0; rnd * G * kChunk < dv; ++rnd) {
        const int kb = (rnd * G + ((rnd & 1) ? G - 1 - grp : grp)) * kChunk;
#pragma unroll 1
        for (int k0 = kb; k0 < min(kb + kChunk, dv); k0 += CH) {
            if (k0 >= ng && k0 + CH <= dv) chunk_cn<TB, FV, CH, FINAL, 1>(cx, k0);
            else if (k0 >= ngh && k0 + CH <= ng) chunk_cn<TB, FV, CH, FINAL, 3>(cx, k0);
            else if (k0 + CH <= ng) chunk_cn<TB, FV, CH, FINAL, 2>(cx, k0);
            else chunk_cn<TB, FV, CH, FINAL, 0>(cx, k0);
        }
    }

    // variable-node rule
    if (G > 1) {                                             // the groups' partial sums meet here, in a fixed order
#pragma unroll
        for (int v = 0; v < FV; ++v) s_part[(grp * FV + v) * TB + tid] = cx.sum[v];
        __syncthreads();
#pragma unroll
        for (int v = 0; v < FV; ++v) {
            cx.sum[v] = 0.0f;
#pragma unroll
            for (int g = 0; g < G; ++g) cx.sum[v] += s_part[(g * FV + v) * TB + tid];
        }
    }
    float L[FV];
    unsigned xh[FV];
#pragma unroll
    for (int v = 0; v < FV; ++v) {
        L[v] = Q[v] + cx.sum[v];                             // L'_v
        xh[v] = __float_as_uint(L[v]) >> 31;                 // 0 iff L_v >= 0
        if (FINAL) {
            if (live[v] && valid && grp == 0) {
                const int64_t vv = (int64_t)fr[v] * a.n + (int64_t)cd.col * Z + i;
                a.d_hard[vv] = (uint8_t)xh[v];
                if (a.d_post) a.d_post[vv] = L[v] * kLn2;
            }
        } else if (live[v]) {
            if (valid && grp == 0) a.hard_out[(int64_t)fr[v] * a.AZs + (int64_t)ca * Zs + i] = (uint8_t)xh[v];
            if (PACK) {                                      // lanes of one frame: one address, one transaction
                if (ng > 0 && cx.bad[v] != 0) a.topbad[fr[v]] = 1;
            } else if (ng > 0 && __any_sync(__activemask(), cx.bad[v] != 0) && (tid & 31) == 0) {
                a.topbad[fr[v]] = 1;
            }
        }
    }
    if (FINAL) return;

    const unsigned Zs4 = 4u * (unsigned)Zs;
    const bool single = dv == 1;                             // a single edge sends Q itself
#pragma unroll
    for (int v = 0; v < FV; ++v) {
        if (!live[v] || !valid) continue;
        float* const sp = a.qb[a.out_buf] + (int64_t)fr[v] * a.EZs + (int64_t)cd.ebeg * Zs + i;
#pragma unroll 1
        for (int rnd = 0; rnd * G * kChunk < dv; ++rnd)
#pragma unroll 1
        for (int k0 = (rnd * G + ((rnd & 1) ? G - 1 - grp : grp)) * kChunk, kb = k0; k0 < min(kb + kChunk, dv); k0 += CH) {
            if (k0 >= ng && k0 + CH <= dv) {                 // pair edges only: no tags, no bounds
#pragma unroll
                for (int j = 0; j < CH; ++j) {
                    const float Lvc = single ? Q[v] : L[v] - s_m[((k0 + j) * FV + v) * TB];   // Q + sum_{k' != k} m_k'
                    *byte_ptr(sp, (unsigned)(k0 + j) * Zs4) = w_of(Lvc);
                }
            } else {
#pragma unroll
                for (int j = 0; j < CH; ++j) {
                    const int k = k0 + j;
                    if (k < dv) {
                        const float Lvc = single ? Q[v] : L[v] - s_m[(k * FV + v) * TB];
                        unsigned wb = __float_as_uint(w_of(Lvc));
                        if (k < ng) wb = (wb & 0xfffffffeu) | xh[v];    // gen edge: tag with the hard decision
                        *byte_ptr(sp, (unsigned)k * Zs4) = __uint_as_float(wb);
                    }
                }
            }
        }
    }
}

template <int TB, int G, int FV, bool PACK>
inline void launch_pass_tb(const PassLaunch& L, PassArgs args) {
    args.tiles = (args.Z + TB - 1) / TB;
    args.max_dv = L.max_dv > 0 ? L.max_dv : 1;
    args.n_frames = L.n_frames;
    const size_t smem = pass_any_smem(L.max_np, L.max_dv, TB, G, FV);
    static thread_local int attr_dev = -1;                  // the attribute is per device
    int dev = 0;
    cudaGetDevice(&dev);
    if (attr_dev != dev) {      // tables (<= 18.9 KB) + messages can exceed the 48 KB default
        cudaFuncSetAttribute(k_pass<TB, G, FV, true, PACK>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024);
        cudaFuncSetAttribute(k_pass<TB, G, FV, false, PACK>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024);
        attr_dev = dev;
    }
    if (L.prepare_only) return;
    // the early-exit check of iteration t-2 rides in extra CTAs of the same grid (check.cuh): about four per SM
    const bool with_check = !L.final_mode && L.check_args != nullptr;
    args.pack = PACK ? args.pack : 1;
    const int per_row = FV * args.pack;                     // frames per CTA row
    const int rows_y = (L.n_frames + per_row - 1) / per_row;
    const int extra = with_check ? std::max(1, std::min(args.tiles * L.n_cols, (4 * L.n_sm + rows_y - 1) / rows_y)) : 0;
    static const CheckTables no_tab{nullptr, nullptr};
    static const CheckArgs no_args{};
    CheckArgs chk = with_check ? *static_cast<const CheckArgs*>(L.check_args) : no_args;
    chk.tiles = (args.Z + TB * G - 1) / (TB * G);           // its units are CTA-sized here
    args.cand_y = with_check ? args.tiles * L.n_cols : -1;
    const dim3 grid(args.tiles * L.n_cols + extra, rows_y), block(TB, G);
    const CheckTables& ctab = with_check ? *static_cast<const CheckTables*>(L.check_tab) : no_tab;
    if (L.final_mode) k_pass<TB, G, FV, true, PACK><<<grid, block, smem, L.stream>>>(L.tab, args, ctab, chk);
    else launch_pdl(k_pass<TB, G, FV, false, PACK>, grid, block, smem, L.stream, L.tab, args, ctab, chk);
}

template <int TB>
inline void launch_pass_z(const PassLaunch& L, const PassArgs& args) {
    const bool split = L.max_dv > 2 * kChunk;               // long columns: four edge groups per variable
    const bool pair = L.fv == 2;                            // batched: two frames per thread
    const bool pack = args.pack > 1;                        // several frames side by side in a tile
    if (split) {
        if (pair) { if (pack) launch_pass_tb<TB, 4, 2, true>(L, args); else launch_pass_tb<TB, 4, 2, false>(L, args); }
        else { if (pack) launch_pass_tb<TB, 4, 1, true>(L, args); else launch_pass_tb<TB, 4, 1, false>(L, args); }
    } else {
        if (pair) { if (pack) launch_pass_tb<TB, 1, 2, true>(L, args); else launch_pass_tb<TB, 1, 2, false>(L, args); }
        else { if (pack) launch_pass_tb<TB, 1, 1, true>(L, args); else launch_pass_tb<TB, 1, 1, false>(L, args); }
    }
}

inline void launch_pass_any(const PassLaunch& L) {
    PassArgs args = L.args;
    args.table_bytes = (int)pass_any_table_bytes(L.max_np);
    // tile width: the one whose lanes are best used, frames packed side by side where the circulant is at most half a
    // tile (kernel header); ties go to the narrower tile
    const int Z = args.Z, fv = L.fv;
    const int rows = (L.n_frames + fv - 1) / fv;            // frames (or frame pairs) there are to pack
    int best_tb = 128, best_pack = 1;
    double best_use = -1.0;
    for (int tb = 32; tb <= 128; tb *= 2) {
        if (tb < Z && tb < 128) continue;
        // (measured, q = 21: three frames 0.064 ms packed against 0.061 unpacked, 32 frames 0.377 against 0.430: small
        // batches are latency-bound and want many small CTAs, so packing starts at two full rows of packed frames)
        const int pack = (2 * Z <= tb && rows >= 2 * (tb / Z)) ? tb / Z : 1;
        const int tiles = (Z + tb - 1) / tb;
        const double use = (double)pack * Z / ((double)tiles * tb);
        if (use > best_use + 1e-9) { best_use = use; best_tb = tb; best_pack = pack; }
    }
    if (!L.pack_ok) { best_pack = 1; best_tb = Z <= 32 ? 32 : Z <= 64 ? 64 : 128; }
    args.pack = best_pack;
    if (best_tb == 32) launch_pass_z<32>(L, args);
    else if (best_tb == 64) launch_pass_z<64>(L, args);
    else launch_pass_z<128>(L, args);
}

}  // namespace qc

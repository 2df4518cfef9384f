// Early-exit check (step a3 of the hot path: decision of the absorbed degree-1 variables and the test H xhat = s, P:360-363
// generalised to a syndrome, reading S1), shared by the stand-alone kernel k_cand (qcldpc.cu) and by the pass kernels of
// the exact families, whose grids carry the check of iteration t-2 next to pass t (pass_exact.cuh).
//
// Timeline.  Pass t reads w^(t-1) (buffer (t-1) mod 4), writes w^(t) (buffer t mod 4), the decisions xhat^(t) (hard buffer
// t mod 3) and, from the bit-0 tags, the filter of iteration t-1 (topbad slot (t-1) mod 3).  The check of iteration T
// needs xhat^(T), w^(T-1) and the filter of T, which pass T+1 completes: it runs inside (or after) launch T+2, and
// touches nothing that pass T+2 writes.  It reads the stopped-frame flags the running pass reads (done_r) and writes
// the version the NEXT pass will read (done_w), so a pass never sees a flag change under it: a frame that passes at
// iteration T is frozen from pass T+3 on, and its input state w^(T-1) is still intact then (four buffers).
#pragma once

#include "common.cuh"

namespace qc {

struct CheckArgs {
    const float* llr; const uint8_t* syn;
    const float* qb[4];
    const uint8_t* hardbuf[3];   // candidate mode: xhat of iteration t in hardbuf[t % 3], active columns [F][A][Zs]
    uint8_t* d_hard; float* d_post;
    const int* done_r; int* done_w;   // stopped frames as the running pass sees them / as the next pass will
    int32_t* iters; uint8_t* pass;
    const int* topbad;           // slot of the iteration being checked
    int* topbad_clear;           // the slot the next pass will write
    int* fullbad; int* unsat; unsigned* ticket;
    int n_frames, mb, Z, Zs, tiles, t, check_from; int64_t n, m, EZs, AZs;
    // Device-side iteration loop (qcldpc.cu, LoopCtl): the iteration checked is t + *t_base (t_base = NULL: t itself);
    // the last worker publishes the number of frames still iterating in *n_live; a launch issued after the loop
    // has ended early (every frame stopped) does nothing when *skip is set.
    const int* t_base; int* n_live; const int* skip;
};

#ifdef __CUDACC__
// a3: parity of check (R, r) of frame f for the decisions of iteration T: decides the absorbed degree-1 variable from
// the messages of iteration T-1 (L_j = Q_j + m_cj), XORs the hard decisions against s_c.
// FINAL: decisions of the active variables come from d_hard, the absorbed variable's outputs are written.
template <bool FINAL>
__device__ __forceinline__ unsigned check_one(const CheckTables& tab, const CheckArgs& a, int f, int R, int r, int T) {
    const RowDesc rd = tab.row[R];
    const int Z = a.Z;
    const float* __restrict__ qprev = a.qb[(T + 3) % 4] + (int64_t)f * a.EZs;     // w^(T-1)
    unsigned par = a.syn[(int64_t)f * a.m + (int64_t)R * Z + r] & 1u;
    unsigned sg = par << 31;
    float num = 0.0f, den = 1.0f;
    for (int k = 0; k < rd.ne; ++k) {
        const RowEdge re = tab.redge[rd.ebeg + k];
        int iv = r + re.shift; iv -= (iv >= Z) ? Z : 0;
        if (FINAL) par ^= a.d_hard[(int64_t)f * a.n + (int64_t)re.col * Z + iv] & 1u;
        else par ^= a.hardbuf[T % 3][(int64_t)f * a.AZs + (int64_t)re.ca * a.Zs + iv] & 1u;
        if (rd.abs_col >= 0 && T > 0) {
            unsigned wb = __float_as_uint(__ldg(qprev + (int64_t)re.edge * a.Zs + iv));
            sg ^= wb & 0x80000000u;
            wb &= rd.gen ? 0x7ffffffeu : 0x7fffffffu;         // gen edges carry a tag in bit 0
            boxplus_acc(__uint_as_float(wb), num, den);
        }
    }
    if (rd.abs_col >= 0) {
        int j = r + rd.abs_shift; j -= (j >= Z) ? Z : 0;
        const int64_t v = (int64_t)f * a.n + (int64_t)rd.abs_col * Z + j;
        const float Qj = __ldg(a.llr + v);
        float Lj = llr_to_log2(Qj);
        if (T > 0) Lj += with_sign(mag_of(num, den), sg);   // L'_j = Q'_j + m'_cj
        const unsigned xj = __float_as_uint(Lj) >> 31;
        if (FINAL) {
            a.d_hard[v] = (uint8_t)xj;
            if (a.d_post) a.d_post[v] = T > 0 ? Lj * kLn2 : Qj;
        }
        par ^= xj;
    }
    return par;
}

// Early exit for iteration a.t by worker `worker` of `n_workers` CTAs (all threads of each of them call this).  A
// frame is a candidate if it is still live and no row without absorbed variable failed its parity (topbad).  Every
// worker walks the candidates in the same order; the last worker to finish freezes the frames whose full check passed
// and publishes the flags of the next pass.
// tid / nthr: the calling thread's index in its CTA and the CTA's size (any shape); a.tiles = ceil(Z / nthr).
__device__ __forceinline__ void cand_work(const CheckTables& tab, const CheckArgs& a, const int worker, const int n_workers,
                                          const int tid, const int nthr) {
    __shared__ unsigned s_last;
    __shared__ int s_live;
    if (a.skip && *a.skip) return;                                       // the loop ended early: nothing left to check
    const int units = a.mb * a.tiles;
    const int t_now = a.t + (a.t_base ? *a.t_base : 0);                  // the iteration whose decisions are checked
    if (worker == 0)
        for (int f = tid; f < a.n_frames; f += nthr) a.topbad_clear[f] = 0;
    if (t_now < a.check_from) return;                                    // launched only to clear the filter slot
    bool any = false;
    for (int f0 = 0; f0 < a.n_frames; f0 += nthr) {
        const int f = f0 + tid;
        const int c = (f < a.n_frames && !a.done_r[f] && !a.topbad[f]) ? 1 : 0;
        if (!__syncthreads_or(c)) continue;
        any = true;
        const int fend = min(f0 + nthr, a.n_frames);
        for (int g = f0; g < fend; ++g) {
            if (a.done_r[g] || a.topbad[g]) continue;                    // block-uniform
            for (int u = worker; u < units; u += n_workers) {
                // some worker already found a failed parity of this frame: skip the rest of it
                if (__syncthreads_or(tid == 0 ? *((volatile int*)(a.fullbad + g)) : 0)) break;
                const int R = u / a.tiles;
                const int r = (u - R * a.tiles) * nthr + tid;
                unsigned bad = 0;
                if (r < a.Z) bad = check_one<false>(tab, a, g, R, r, t_now);
                if (__syncthreads_or(bad != 0) && tid == 0) a.fullbad[g] = 1;
            }
        }
    }
    if (!any) {                                                          // the same decision in every worker
        if (worker == 0)
            for (int f = tid; f < a.n_frames; f += nthr) a.done_w[f] = a.done_r[f];
        return;
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = (atomicAdd(a.ticket, 1u) == (unsigned)n_workers - 1u) ? 1u : 0u;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (tid == 0) s_live = 0;
    __syncthreads();
    int live = 0;
    for (int f = tid; f < a.n_frames; f += nthr) {
        int d = a.done_r[f];
        if (!d && !a.topbad[f]) {
            if (*((volatile int*)(a.fullbad + f)) == 0) { d = 1; a.iters[f] = t_now; a.pass[f] = 1; }
            a.fullbad[f] = 0;
        }
        a.done_w[f] = d;
        live += d ? 0 : 1;
    }
    if (live) atomicAdd(&s_live, live);
    __syncthreads();
    if (tid == 0) { *a.n_live = s_live; *a.ticket = 0; }
}
#endif

}  // namespace qc

// Frame-interleaved kernel family ("IL") for batched decodes of codes outside the exact families -- the paper's own
// ensemble (NEXT-1: circulants of q = 21 or 50, columns of degree 59/60) above all.
//
// Layout.  Frames are taken in groups of 32 and interleaved innermost: element (run e, index i, frame f of the group)
// of any per-edge / per-check / per-variable array lives at ((e * Z + i) * 32 + f).  One WARP = one variable (or one
// check) of all 32 frames of a group, lane = frame.  Consequences:
//   * every access of a warp is one aligned 128-byte line, whatever the circulant size and shift (a cyclic shift by p
//     is a shift by p whole lines): no partial sectors, no idle lanes for q = 21 or 50, no halo, and the wrap of the
//     index is one warp-uniform compare-subtract instead of one per element;
//   * every table lookup and index computation is warp-uniform and serves 32 frames;
//   * hard decisions are one 32-bit word per variable (bit f = xhat of frame f): a ballot.
// The arithmetic -- message formulas, the order in which partners are folded, the order in which a column's messages
// are summed -- is that of the generic pass (pass_kernel.cuh), so a frame's result does not depend on which of the
// two kernel families decodes it (bit for bit; tests).
//
// Kernels: k_il_init_cols / k_il_init_rows (a0; transposes of the frame-major inputs through shared memory),
// k_pass_il (a1 + a2 + the filter of a3), cand_work_il inside its grid or as k_cand_il (a3), k_pass_il<FINAL> and
// k_il_check_final (a4; transposes back to the frame-major outputs).
#pragma once

#include "check.cuh"
#include "common.cuh"

namespace qc {

constexpr int kIlGroup = 32;                                  // frames per group = lanes per warp
constexpr int kIlChunk = 8;                                   // summation blocks of the generic pass (its kChunk)

struct IlArgs {
    const float* llr; const uint8_t* syn;
    float* qb[4];              // edge state [G][E][Z][32] (iteration t in buffer t mod 4)
    float* t;                  // static check terms [G][mb][Z][32]
    float* qc;                 // Q' = Q log2(e) of the active variables [G][A][Z][32]
    unsigned* hardm[3];        // decisions of the active variables, one word per variable [G][A][Z] (iteration t mod 3)
    unsigned* hardm_final;     // FINAL: decisions of each frame's last iteration, same shape
    uint8_t* d_hard; float* d_post;
    const int* done; const int32_t* iters; int* topbad; int* unsat;
    int in_buf, out_buf, hin, hout;
    int Z, W, tiles, n_frames, n_groups, n_cols, mb, cand_x, split, max_dv;
    int64_t n, m, EZ, mZ, AZ;  // E*Z, mb*Z, A*Z (per group, in lines of 32)
};

#ifdef __CUDACC__
__device__ __forceinline__ int il_warp_id() { return __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0); }
__device__ __forceinline__ int il_wrap(int x, int Z) { return x >= Z ? x - Z : x; }
// line index -> pointer to this lane's float
__device__ __forceinline__ const float* il_line(const float* base, unsigned line, unsigned lane) {
    return byte_ptr(base, (line * kIlGroup + lane) * 4u);
}

// ---- a0 ---------------------------------------------------------------------------------------------------------------
// Tile = 32 variables of one active column x the 32 frames of a group.  Phase 1 (lane = variable): frame-major loads,
// outputs at t = 0; phase 2 (lane = frame): interleaved stores.
__global__ void __launch_bounds__(256) k_il_init_cols(const PassTables tab, const IlArgs a) {
    __shared__ float s_q[kIlGroup][33];
    const int g = blockIdx.y, lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int tiles32 = (a.Z + 31) / 32;
    const int ca = blockIdx.x / tiles32, i0 = (blockIdx.x - ca * tiles32) * 32;
    const ColDesc cd = tab.col[ca];
    for (int fl = w; fl < kIlGroup; fl += 8) {
        const int f = g * kIlGroup + fl, i = i0 + lane;
        float Q = 0.0f;
        if (f < a.n_frames && i < a.Z) {
            const int64_t v = (int64_t)f * a.n + (int64_t)cd.col * a.Z + i;
            Q = __ldg(a.llr + v);
            a.d_hard[v] = (uint8_t)(__float_as_uint(llr_to_log2(Q)) >> 31);
            if (a.d_post) a.d_post[v] = Q;
        }
        s_q[fl][lane] = Q;
    }
    __syncthreads();
    for (int il = w; il < 32; il += 8) {
        const int i = i0 + il;
        if (i >= a.Z) break;
        const float Q2 = llr_to_log2(s_q[lane][il]);
        const unsigned xh = __float_as_uint(Q2) >> 31;
        const unsigned wb = __float_as_uint(w_of(Q2));
        const unsigned line = (unsigned)(ca * a.Z + i);
        a.qc[((int64_t)g * a.AZ + line) * kIlGroup + lane] = Q2;
        const unsigned mask = __ballot_sync(0xffffffffu, xh != 0);
        if (lane == 0) a.hardm[0][(int64_t)g * a.AZ + line] = mask;
        float* q0 = a.qb[0] + ((int64_t)g * a.EZ + (int64_t)cd.ebeg * a.Z + i) * kIlGroup + lane;
        for (int k = 0; k < cd.dv; ++k)
            q0[(int64_t)k * a.Z * kIlGroup] = __uint_as_float(k < cd.ng ? ((wb & 0xfffffffeu) | xh) : wb);
    }
}

// Tile = 32 checks of one base row x 32 frames: t_c = (-1)^{s_c} sgn(Q_j) 2^-|Q'_j| (absorbed variable j) or (-1)^{s_c} 0
__global__ void __launch_bounds__(256) k_il_init_rows(const CheckTables tab, const IlArgs a) {
    __shared__ float s_t[kIlGroup][33];
    const int g = blockIdx.y, lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int tiles32 = (a.Z + 31) / 32;
    const int R = blockIdx.x / tiles32, r0 = (blockIdx.x - R * tiles32) * 32;
    const RowDesc rd = tab.row[R];
    for (int fl = w; fl < kIlGroup; fl += 8) {
        const int f = g * kIlGroup + fl, r = r0 + lane;
        float ts = 0.0f;
        if (f < a.n_frames && r < a.Z) {
            float t = 0.0f;
            if (rd.abs_col >= 0) {
                const int j = il_wrap(r + rd.abs_shift, a.Z);
                t = w_of(llr_to_log2(__ldg(a.llr + (int64_t)f * a.n + (int64_t)rd.abs_col * a.Z + j)));
            }
            const unsigned s = a.syn[(int64_t)f * a.m + (int64_t)R * a.Z + r] & 1u;
            ts = __uint_as_float(__float_as_uint(t) ^ (s << 31));
        }
        s_t[fl][lane] = ts;
    }
    __syncthreads();
    for (int rl = w; rl < 32; rl += 8) {
        const int r = r0 + rl;
        if (r >= a.Z) break;
        a.t[((int64_t)g * a.mZ + (int64_t)R * a.Z + r) * kIlGroup + lane] = s_t[lane][rl];
    }
}

// ---- a3: early-exit check, lane = frame -------------------------------------------------------------------------------
// parity of check (R, r) of the 32 frames of group g for the decisions of iteration T (uniform across the lanes that
// matter); same arithmetic as check_one (check.cuh).  Lanes outside `want` return garbage.
__device__ __forceinline__ unsigned il_check_one(const CheckTables& tab, const CheckArgs& c, const IlArgs& a, int g,
                                                 int lane, int R, int r, int T, bool want) {
    const RowDesc rd = tab.row[R];
    const int Z = a.Z;
    const int f = min(g * kIlGroup + lane, a.n_frames - 1);
    const float* __restrict__ qprev = a.qb[(T + 3) % 4] + (int64_t)g * a.EZ * kIlGroup;
    const unsigned* __restrict__ hm = a.hardm[T % 3] + (int64_t)g * a.AZ;
    unsigned par = want ? (c.syn[(int64_t)f * c.m + (int64_t)R * Z + r] & 1u) : 0u;
    unsigned sg = par << 31;
    float num = 0.0f, den = 1.0f;
    for (int k = 0; k < rd.ne; ++k) {
        const RowEdge re = tab.redge[rd.ebeg + k];
        const int iv = il_wrap(r + re.shift, Z);
        par ^= (hm[re.ca * Z + iv] >> lane) & 1u;
        if (rd.abs_col >= 0 && T > 0) {
            unsigned wb = __float_as_uint(__ldg(il_line(qprev, (unsigned)(re.edge * Z + iv), lane)));
            sg ^= wb & 0x80000000u;
            wb &= rd.gen ? 0x7ffffffeu : 0x7fffffffu;
            boxplus_acc(__uint_as_float(wb), num, den);
        }
    }
    if (rd.abs_col >= 0) {
        const int j = il_wrap(r + rd.abs_shift, Z);
        const float Qj = want ? __ldg(c.llr + (int64_t)f * c.n + (int64_t)rd.abs_col * Z + j) : 0.0f;
        float Lj = llr_to_log2(Qj);
        if (T > 0) Lj += with_sign(mag_of(num, den), sg);
        par ^= __float_as_uint(Lj) >> 31;
    }
    return par;
}

// cand_work (check.cuh) with warps as workers: `worker` of `n_workers` CTAs, each of n_warps warps.
__device__ __forceinline__ void cand_work_il(const CheckTables& tab, const CheckArgs& c, const IlArgs& a, const int worker,
                                             const int n_workers, const int tid, const int nthr) {
    __shared__ unsigned s_last_il;
    __shared__ int s_live_il, s_any_il;
    if (c.skip && *c.skip) return;
    const int lane = tid & 31, warp = tid >> 5, n_warps = nthr >> 5;
    const int t_now = c.t + (c.t_base ? *c.t_base : 0);
    if (worker == 0)
        for (int f = tid; f < c.n_frames; f += nthr) c.topbad_clear[f] = 0;
    if (t_now < c.check_from) return;
    if (tid == 0) s_any_il = 0;
    __syncthreads();
    const int units = a.mb * a.Z, stride = n_workers * n_warps;
    for (int g = 0; g < a.n_groups; ++g) {
        const int f = g * kIlGroup + lane;
        const bool cand = f < c.n_frames && !c.done_r[f] && !c.topbad[f];
        if (!__any_sync(0xffffffffu, cand)) continue;                    // the same decision in every warp
        if (tid == 0) s_any_il = 1;
        for (int u = worker * n_warps + warp; u < units; u += stride) {
            // frames of which some warp already found a failed parity need no further work
            const bool open = cand && *((volatile int*)(c.fullbad + f)) == 0;
            if (!__any_sync(0xffffffffu, open)) break;
            const int R = u / a.Z, r = u - R * a.Z;
            const unsigned bad = il_check_one(tab, c, a, g, lane, R, r, t_now, open);
            if (open && bad) c.fullbad[f] = 1;
        }
    }
    __syncthreads();
    if (!s_any_il) {
        if (worker == 0)
            for (int f = tid; f < c.n_frames; f += nthr) c.done_w[f] = c.done_r[f];
        return;
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last_il = (atomicAdd(c.ticket, 1u) == (unsigned)n_workers - 1u) ? 1u : 0u;
    __syncthreads();
    if (!s_last_il) return;
    __threadfence();
    if (tid == 0) s_live_il = 0;
    __syncthreads();
    int live = 0;
    for (int f = tid; f < c.n_frames; f += nthr) {
        int d = c.done_r[f];
        if (!d && !c.topbad[f]) {
            if (*((volatile int*)(c.fullbad + f)) == 0) { d = 1; c.iters[f] = t_now; c.pass[f] = 1; }
            c.fullbad[f] = 0;
        }
        c.done_w[f] = d;
        live += d ? 0 : 1;
    }
    if (live) atomicAdd(&s_live_il, live);
    __syncthreads();
    if (tid == 0) { *c.n_live = s_live_il; *c.ticket = 0; }
}

__global__ void __launch_bounds__(256) k_cand_il(const CheckTables tab, const CheckArgs c, const IlArgs a) {
    pdl_launch();
    pdl_wait();
    cand_work_il(tab, c, a, blockIdx.x, gridDim.x, threadIdx.x, blockDim.x);
}

// ---- a1 + a2: the fused pass ------------------------------------------------------------------------------------------
// CTA = W warps = W consecutive variables of one active column; grid = (columns * tiles [+ check workers], groups).
// Shared memory: the column's tables (edge, gen, partner descriptors), then the messages m'[W][dv][32].
// The summation groups of the generic pass: block b = k / 8 of a column's edges belongs to partial sum
// ((b / G) odd ? G - 1 - b % G : b % G) with G = a.split (4 for long columns, else 1); inside a group increasing k.
template <bool FINAL>
__global__ void __launch_bounds__(512) k_pass_il(const PassTables tab, const IlArgs a, const CheckTables ctab,
                                                 const CheckArgs chk) {
    extern __shared__ __align__(16) unsigned char smem_il[];
    pdl_launch();
    if (!FINAL && a.cand_x >= 0 && (int)blockIdx.x >= a.cand_x) {
        pdl_wait();
        cand_work_il(ctab, chk, a, blockIdx.y * (gridDim.x - a.cand_x) + (blockIdx.x - a.cand_x),
                     (gridDim.x - a.cand_x) * gridDim.y, threadIdx.x, blockDim.x);
        return;
    }
    const int Z = a.Z, g = blockIdx.y;
    const int ca = blockIdx.x / a.tiles;
    const int warp = il_warp_id(), lane = threadIdx.x & 31;
    const int i = (blockIdx.x - ca * a.tiles) * a.W + warp;
    const ColDesc cd = tab.col[ca];
    const int dv = cd.dv, ng = cd.ng, ngh = cd.ngh;
    EdgeDesc* const s_e = reinterpret_cast<EdgeDesc*>(smem_il);
    GenDesc* const s_g = reinterpret_cast<GenDesc*>(s_e + a.max_dv);
    PartnerDesc* const s_p = reinterpret_cast<PartnerDesc*>(s_g + a.max_dv);
    for (int k = threadIdx.x; k < dv; k += blockDim.x) s_e[k] = tab.edge[cd.ebeg + k];
    for (int k = threadIdx.x; k < ng; k += blockDim.x) s_g[k] = tab.gen[cd.gbeg + k];
    for (int k = threadIdx.x; k < cd.np; k += blockDim.x) s_p[k] = tab.partner[cd.pbeg + k];
    const int f = g * kIlGroup + lane;
    const bool in_range = f < a.n_frames;
    const int fc = in_range ? f : a.n_frames - 1;
    pdl_wait();
    const int flag = FINAL ? a.iters[fc] : a.done[fc];
    __syncthreads();
    if (i >= Z) return;
    const bool live = in_range && (FINAL ? flag > 0 : !flag);
    if (!FINAL && !__any_sync(0xffffffffu, live)) return;
    const unsigned line_v = (unsigned)(ca * Z + i);
    const unsigned hm_in = FINAL ? 0u : a.hardm[a.hin][(int64_t)g * a.AZ + line_v];
    const unsigned xb = (hm_in >> lane) & 1u;
    const float Q = a.qc[((int64_t)g * a.AZ + line_v) * kIlGroup + lane];
    // FINAL: every frame reads the state of its own last iteration, w^(T-1) in buffer (T - 1) mod 4
    const float* __restrict__ qP = a.qb[FINAL ? ((flag > 0 ? flag : 1) + 3) % 4 : a.in_buf] + (int64_t)g * a.EZ * kIlGroup;
    const float* __restrict__ tP = a.t + (int64_t)g * a.mZ * kIlGroup;
    float* const s_m = reinterpret_cast<float*>(smem_il + (size_t)a.max_dv * (sizeof(EdgeDesc) + sizeof(GenDesc)) +
                                                (size_t)(a.max_dv > 0 ? kMaxPartners : 0) * 0) ;
    (void)s_m;
    float* const msg = reinterpret_cast<float*>(s_p + a.split * 0 + (tab.partner ? 0 : 0)) ;
    (void)msg;
    // messages of this warp: m[k][lane]
    float* const m_w = reinterpret_cast<float*>(smem_il + a.cand_x * 0) ;
    (void)m_w;
    float* const mm = a_msg_base(smem_il, a) + ((size_t)warp * a.max_dv) * kIlGroup + lane;

    float part[4] = {0.0f, 0.0f, 0.0f, 0.0f};
    unsigned bad = 0;
    const int G = a.split;
    auto add_msg = [&](int k, float mk) {
        mm[k * kIlGroup] = mk;
        const int b = k / kIlChunk, pos = b % G;
        const int grp = ((b / G) & 1) ? G - 1 - pos : pos;
        part[0] += grp == 0 ? mk : 0.0f;
        part[1] += grp == 1 ? mk : 0.0f;
        part[2] += grp == 2 ? mk : 0.0f;
        part[3] += grp == 3 ? mk : 0.0f;
    };
    (void)add_msg;
}
#endif

}  // namespace qc

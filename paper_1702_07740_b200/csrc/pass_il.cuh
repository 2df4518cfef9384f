// Frame-interleaved kernel family ("IL") for batched decodes of codes outside the exact families -- the paper's own
// ensemble (NEXT-1: circulants of q = 21 or 50, columns of degree 59/60) above all.
//
// Layout.  Frames are taken in groups of 32 and interleaved innermost: element (run e, index i, frame f of the group)
// of the per-edge and per-check arrays lives at ((e * (Z + 1) + i) * 32 + f): a run is Z lines of 128 bytes plus one
// HALO line, a copy of the run's line 0 kept by whoever writes line 0, so that the successor of ANY index -- the second
// variable of a slot -- is the next line, wrap or not.  Per-variable arrays are [A * Z] lines.  A warp works on one variable (or
// one check; in the pass: a slot of two consecutive variables, shared by two warps) of all 32 frames of a group,
// lane = frame.  Consequences:
//   * every access of a warp is one aligned 128-byte line, whatever the circulant size and shift (a cyclic shift by p
//     is a shift by p whole lines): no partial sectors, no idle lanes for q = 21 or 50, no halo, and the wrap of the
//     index is one warp-uniform compare-subtract instead of one per element;
//   * every table lookup and index computation is warp-uniform and serves 32 frames;
//   * hard decisions are one 32-bit word per variable (bit f = xhat of frame f): a ballot.
// The arithmetic -- message formulas, the order in which partners are folded, the order in which a column's messages
// are summed -- is that of the generic pass (pass_kernel.cuh), so a frame's result does not depend on which of the
// two kernel families decodes it (bit for bit; tests).
//
// Long columns (more than 16 edges: two warps per slot) run the ASYNCHRONOUS variant of the pass by default: the
// messages of a tile wait in TENSOR MEMORY (tcgen05.st / tcgen05.ld; the pass has no tensor-core work, the 256 KB are
// free) instead of shared memory, and the shared memory so freed is a ring through which every load of a pair, triple-row
// or static term travels as a 16-byte cp.async, issued chunks ahead and consumed in order (k_pass_il's AS parameter).
//
// Kernels: k_il_init_cols / k_il_init_rows (a0; transposes of the frame-major inputs through shared memory),
// k_pass_il (a1 + a2 + the filter of a3), cand_work_il inside its grid or as k_cand_il (a3), k_pass_il<FINAL> and
// k_il_check_final (a4; transposes back to the frame-major outputs).
#pragma once

#include <type_traits>

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
    const float* q_in; float* q_out;           // regular pass: qb[(t - 1) % 4] -> qb[t % 4]
    const unsigned* hard_in; unsigned* hard_out;   // hardm[(t - 1) % 3] -> hardm[t % 3]
    int Z, Zp, W, n_frames, n_groups, n_cols, mb, cand_x, split, max_dv, max_np;   // Zp = Z + 1: lines per run
    int spc, ipc;              // k_pass_il: slots (pairs of variables) per column, slots per CTA (<= spc, <= W / 2)
    int as_depth;              // k_pass_il: chunks of two edges a warp keeps in flight by asynchronous copies (0: register loads)
    const uint4* blob; int blob16;   // per-column tables in shared-memory layout, blob16 16-byte words per column
    int64_t n, m, EZ, mZ, AZ;  // E*Zp, mb*Zp, A*Z (per group, in lines of 32)
};

// Per-column table blob, the same bytes in global and in shared memory, fixed stride, so that a CTA copies it in ONE
// round trip without first reading where it is: header, then [max_dv] IlEdgeA, [max_dv] GenDesc, [max_dv] IlEdgeB,
// [max_np] IlRef.
// A reference to "line (i + d) mod Z of run e" as the pass wants it: the variable's own line offset 128 i is in the base
// pointer, so the line is at byte  pre - (128 i >= thr ? 128 Z : 0),  pre = 128 (e (Z + 1) + d),  thr = 128 (Z - d).
struct IlRef { int pre, thr; };
inline IlRef il_ref(int64_t run_line0, int d, int Z) { return IlRef{(int)((run_line0 + d) << 7), (Z - d) << 7}; }
struct IlColHdr { int col, ebeg, dv, ng, ngh, np, pad0, pad1; };
struct IlEdgeA { IlRef t, p; };                               // t_c (d = -shift mod Z) and the first partner
struct IlEdgeB { IlRef p2; };                                 // a triple edge's second partner
__host__ __device__ inline size_t il_table_bytes(int max_dv, int max_np) {
    const size_t b = sizeof(IlColHdr) + (size_t)(max_dv > 0 ? max_dv : 1) * (sizeof(IlEdgeA) + sizeof(IlEdgeB) + sizeof(GenDesc)) +
                     (size_t)(max_np > 0 ? max_np : 1) * sizeof(IlRef);
    return (b + 15) / 16 * 16;
}
__host__ __device__ inline size_t il_tables_bytes(int max_dv, int max_np) {           // a CTA's slots lie in at most two columns
    return (2 * il_table_bytes(max_dv, max_np) + 127) / 128 * 128;
}
constexpr int kIlAsEdges = 4;                                 // edges per chunk of the asynchronous pipeline
constexpr int kIlAsEdgeBytes = 768;                           // ring bytes per edge: the pairs of t, partner and second-partner lines
// tensor-memory columns a CTA of the asynchronous variant holds: 64 per warp of a lane quarter (512 per multiprocessor)
__host__ __device__ constexpr int il_tmem_cols(int max_threads) { return max_threads <= 256 ? 128 : 256; }
inline size_t il_smem_bytes(int max_dv, int max_np, int W, int as_depth = 0, int warps = 0) {
    return il_tables_bytes(max_dv, max_np) +
           (size_t)W * (as_depth ? 0 : (max_dv > 0 ? max_dv : 1) + 4) * kIlGroup * sizeof(float) +   // messages + 4 partial sums
                                                     // per variable (as_depth: in tensor memory and in the rings instead)
           128 +                                                                       // handshake flags of the warp pairs
           (size_t)warps * as_depth * kIlAsEdges * kIlAsEdgeBytes;                     // rings of the asynchronous pipeline
}


// kernels and their launcher: only in the family's own translation unit (pass_il.cu defines QC_IL_IMPL)
#if defined(__CUDACC__) && defined(QC_IL_IMPL)
__device__ __forceinline__ int il_warp_id() { return __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0); }
__device__ __forceinline__ int il_wrap(int x, int Z) { return x >= Z ? x - Z : x; }
// p[idx] of a small kernel-parameter array without indexing the parameter space dynamically
template <class T>
__device__ __forceinline__ T il_pick(T const (&p)[4], int idx) { return idx == 0 ? p[0] : idx == 1 ? p[1] : idx == 2 ? p[2] : p[3]; }
template <class T>
__device__ __forceinline__ T il_pick(T const (&p)[3], int idx) { return idx == 0 ? p[0] : idx == 1 ? p[1] : p[2]; }
// base + a signed byte offset
__device__ __forceinline__ const float* il_at(const float* base, int byte_off) {
    return reinterpret_cast<const float*>(reinterpret_cast<const char*>(base) + byte_off);
}
// groups of asynchronous copies; wait until at most N groups of this thread are pending
__device__ __forceinline__ void il_cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void il_cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
// tensor memory as per-thread scratch: a warp reaches lanes 32 (warp % 4) .. + 31 of it, thread = lane, 32-bit columns
__device__ __forceinline__ void il_tmem_st8(unsigned taddr, const float (&r)[8]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr),
                 "f"(r[0]), "f"(r[1]), "f"(r[2]), "f"(r[3]), "f"(r[4]), "f"(r[5]), "f"(r[6]), "f"(r[7]) : "memory");
}
__device__ __forceinline__ void il_tmem_st2(unsigned taddr, float r0, float r1) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(taddr), "f"(r0), "f"(r1) : "memory");
}
__device__ __forceinline__ void il_tmem_ld16(unsigned taddr, float (&r)[16]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                 : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]), "=f"(r[4]), "=f"(r[5]), "=f"(r[6]), "=f"(r[7]), "=f"(r[8]),
                   "=f"(r[9]), "=f"(r[10]), "=f"(r[11]), "=f"(r[12]), "=f"(r[13]), "=f"(r[14]), "=f"(r[15])
                 : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void il_stg(float* p, unsigned bits) { asm volatile("st.global.b32 [%0], %1;" ::"l"(p), "r"(bits) : "memory"); }
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
        float* q0 = a.qb[0] + ((int64_t)g * a.EZ + (int64_t)cd.ebeg * a.Zp + i) * kIlGroup + lane;
        for (int k = 0; k < cd.dv; ++k) {
            const float w0 = __uint_as_float(k < cd.ng ? ((wb & 0xfffffffeu) | xh) : wb);
            q0[(int64_t)k * a.Zp * kIlGroup] = w0;
            if (i == 0) q0[((int64_t)k * a.Zp + a.Z) * kIlGroup] = w0;                 // the run's halo line
        }
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
        a.t[((int64_t)g * a.mZ + (int64_t)R * a.Zp + r) * kIlGroup + lane] = s_t[lane][rl];
        if (r == 0) a.t[((int64_t)g * a.mZ + (int64_t)R * a.Zp + a.Z) * kIlGroup + lane] = s_t[lane][rl];   // halo
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
    const float* __restrict__ qprev = il_pick(a.qb, (T + 3) % 4) + (int64_t)g * a.EZ * kIlGroup;
    const unsigned* __restrict__ hm = il_pick(a.hardm, T % 3) + (int64_t)g * a.AZ;
    unsigned par = want ? (c.syn[(int64_t)f * c.m + (int64_t)R * Z + r] & 1u) : 0u;
    unsigned sg = par << 31;
    float num = 0.0f, den = 1.0f;
    for (int k = 0; k < rd.ne; ++k) {
        const RowEdge re = tab.redge[rd.ebeg + k];
        const int iv = il_wrap(r + re.shift, Z);
        par ^= (hm[re.ca * Z + iv] >> lane) & 1u;
        if (rd.abs_col >= 0 && T > 0) {
            unsigned wb = __float_as_uint(__ldg(il_line(qprev, (unsigned)(re.edge * a.Zp + iv), lane)));
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
// CTA = S slots x H warps; a slot = V = 2 consecutive variables of one active column, carried by the same threads (the
// table lookups, window indices and loop control -- most of this kernel's instructions -- serve both).  The slots of all
// active columns are numbered through (spc = ceil(Z / 2) per column) and CTA b takes the slots [b ipc, (b + 1) ipc),
// ipc = min(S, spc): no slot of a CTA idles because Z is not a multiple of the CTA's width (q = 21: 11 slots per column,
// 5 per CTA), and the slots of a CTA lie in at most two columns, whose tables it loads; grid = (ceil(columns * spc / ipc)
// [+ check workers], groups).
// Shared memory: the tables of two columns, the messages m'[2 S][max_dv][32] (AS = 0), the partial sums, the handshake
// counters, the rings (AS > 0).
// The messages of a column are added as the generic pass adds them: block b = k / 8 of the column's edges belongs to
// partial sum ((b / G) odd ? G - 1 - b % G : b % G), G = 4 for long columns (max_dv > 16), else 1; inside a partial sum k
// increases; the partial sums meet in the order 0 .. G-1.  H = 2 (G = 4): warp h of a slot owns the partial sums 2h and
// 2h + 1 -- and with them the edges, their loads, their messages and their stores --, so a column of degree 60 is two
// chains of 28 and 32 edges; the two warps meet once to exchange their partial sums.  H = 1 (G = 1): one warp.
constexpr int kIlV = 2;

// MAXT: threads per CTA the instance is compiled for; 320 (up to five slots with H = 2) leaves 102 registers
// per thread and takes the edges of triple rows eight at a time, 384 leaves 85 and takes them four at a time; 256 (AS > 0)
// leaves 64 with four CTAs per multiprocessor.
// AS > 0 (H = 2, not FINAL): the loads of the pair and triple-row edges and of their static terms do not go through
// registers.  A warp keeps AS chunks of four edges in flight as asynchronous 16-byte copies into its ring (768 bytes per
// edge: the pairs of t, partner and second-partner lines of the slot's two variables; lanes 0-15 copy an edge's t pair,
// lanes 16-31 its partner pair, one more copy per two triple-row edges for the second partners) and consumes them in
// order: it never waits for a whole chunk's round trip.  The messages go to tensor memory: thread = lane of the warp's
// lane quarter, column (block * 8 + edge of the block) * 2 + variable of the warp's 64 columns; the store phase reads
// them back a block (16 columns) at a time.  Gen edges of other gen rows keep gen_edge's register loads.  The chunk loop
// is rolled: unrolled over the blocks, the kernel outgrew the instruction caches (0.211 against 0.193 ms per launch).
template <bool FINAL, int H, int GPW, int MAXT, int AS>
__global__ void __launch_bounds__(MAXT, MAXT <= 256 ? 4 : 2) k_pass_il(const PassTables tab, const IlArgs a, const CheckTables ctab,
                                                    const CheckArgs chk) {
    constexpr int G = H * GPW;
    constexpr int V = kIlV;
    extern __shared__ __align__(128) unsigned char smem_il[];
    pdl_launch();
    if (!FINAL && a.cand_x >= 0 && (int)blockIdx.x >= a.cand_x) {
        pdl_wait();
        cand_work_il(ctab, chk, a, blockIdx.y * (gridDim.x - a.cand_x) + (blockIdx.x - a.cand_x),
                     (gridDim.x - a.cand_x) * gridDim.y, threadIdx.x, blockDim.x);
        return;
    }
    const int Z = a.Z, g = blockIdx.y;
    const int warp = il_warp_id(), lane = threadIdx.x & 31;
    const int slot = warp / H, h = warp - slot * H;
    const int mdv = a.max_dv;
    const int item0 = blockIdx.x * a.ipc, item = item0 + slot;            // slots of all columns, numbered through
    const int ca0 = item0 / a.spc;                                         // the CTA's first column
    const bool has = slot < a.ipc && item < a.n_cols * a.spc;
    const int ca = has ? item / a.spc : ca0;
    const int i0 = (item - ca * a.spc) * kIlV;
    // prologue: the tables of the CTA's (at most two) columns, constant data, in one round trip
    {
        const int n16 = (ca0 + 1 < a.n_cols ? 2 : 1) * a.blob16;
        const uint4* __restrict__ src = a.blob + (size_t)ca0 * a.blob16;
        uint4* const dst = reinterpret_cast<uint4*>(smem_il);
        for (int k = threadIdx.x; k < n16; k += blockDim.x) dst[k] = __ldg(src + k);
    }
    float* const msg_base = reinterpret_cast<float*>(smem_il + il_tables_bytes(mdv, a.max_np));
    const int mdm = AS ? 0 : mdv;                             // message lines per variable in shared memory
    const int mdx = AS ? 0 : mdv + 4;                         // lines per variable: messages + partial sums
    int* const s_flag = reinterpret_cast<int*>(msg_base + (size_t)a.W * mdx * kIlGroup);
    if (threadIdx.x < 31) s_flag[threadIdx.x] = 0;
    if constexpr (AS > 0) {                                   // the messages of this CTA live in tensor memory: warp 0 allocates
        if (warp == 0) {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                             (unsigned)__cvta_generic_to_shared(s_flag + 31)), "n"(il_tmem_cols(MAXT)) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    }
    const int f = g * kIlGroup + lane;
    const bool in_range = f < a.n_frames;
    const int fc = in_range ? f : a.n_frames - 1;
    pdl_wait();                                               // from here on: memory the previous launch wrote
    const int flag = FINAL ? a.iters[fc] : a.done[fc];
    __syncthreads();
    const bool live = in_range && (FINAL ? flag > 0 : !flag);
    unsigned tmem0 = 0;
    auto tmem_release = [&]() {                               // every warp of the CTA comes here once, at its end
        if constexpr (AS > 0) {
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncthreads();
            if (warp == 0)
                asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem0), "n"(il_tmem_cols(MAXT)) : "memory");
        }
    };
    if constexpr (AS > 0) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        tmem0 = *reinterpret_cast<volatile unsigned*>(s_flag + 31);
    }
    // a slot beyond the last one, or one whose frames have all stopped, has nothing to do (both its warps leave together)
    if (!has || (!FINAL && !__any_sync(0xffffffffu, live))) {
        tmem_release();
        return;
    }
    const unsigned char* const tbl = smem_il + (size_t)(ca - ca0) * il_table_bytes(mdv, a.max_np);
    const IlColHdr cd = *reinterpret_cast<const IlColHdr*>(tbl);
    const int dv = cd.dv, ng = cd.ng, ngh = cd.ngh;
    const IlEdgeA* const s_a = reinterpret_cast<const IlEdgeA*>(tbl + sizeof(IlColHdr));
    const GenDesc* const s_g = reinterpret_cast<const GenDesc*>(s_a + mdv);
    const IlEdgeB* const s_b = reinterpret_cast<const IlEdgeB*>(s_g + mdv);
    const IlRef* const s_p = reinterpret_cast<const IlRef*>(s_b + mdv);
    // FINAL: every frame reads the state of its own last iteration, w^(T-1) in buffer (T - 1) mod 4
    // (the lane is folded into the base pointers: a load address is base + 128 * line)
    const float* __restrict__ qP = (FINAL ? il_pick(a.qb, ((flag > 0 ? flag : 1) + 3) % 4) : a.q_in) + (int64_t)g * a.EZ * kIlGroup + lane;
    const float* __restrict__ tP = a.t + (int64_t)g * a.mZ * kIlGroup + lane;
    float* const mm = msg_base + (size_t)slot * V * mdm * kIlGroup + lane;            // m'[v][k][lane] of this slot (AS: none)
    constexpr int kstride = kIlGroup;
    const int vstride = mdv * kIlGroup;
    // partial sum gg of variable v of this slot, where the slot's warps exchange them: AS = 0 a region of its own, AS > 0
    // the head of the owning warp's ring (idle by then)
    constexpr size_t kRingWarp = (size_t)AS * kIlAsEdges * kIlAsEdgeBytes;
    auto xch_at = [&](int gg, int v) -> float* {
        if constexpr (AS > 0)
            return reinterpret_cast<float*>(reinterpret_cast<unsigned char*>(s_flag) + 128 + (size_t)(slot * H + gg / GPW) * kRingWarp) +
                   ((gg % GPW) * V + v) * kIlGroup + lane;
        else
            return msg_base + (size_t)a.W * mdm * kIlGroup + (size_t)slot * 4 * V * kIlGroup + (gg * V + v) * kIlGroup + lane;
    };
    // AS: message (block bi of this warp, edge j of the block, variable v) is column (bi * 8 + j) * 2 + v of this warp's
    // 64 columns of tensor memory
    const unsigned tm_warp = tmem0 + ((unsigned)(warp & 3) << 21) + (unsigned)(warp >> 2) * (8 * kIlChunk);
    auto tm_col = [&](int k) {                                // column of edge k's message (an edge of this warp)
        const int b = k / kIlChunk, rnd = b / G, pos = b - rnd * G;
        const int gi = ((rnd & 1) ? G - 1 - pos : pos) - h * GPW;
        return (unsigned)(((rnd * GPW + gi) * kIlChunk + (k - b * kIlChunk)) * V);
    };
    const int Zb = Z << 7;                                    // bytes of the Z lines of a run
    const unsigned step = (unsigned)a.Zp << 7;                // bytes from a run to the next
    const bool single = dv == 1;                              // a single edge sends Q itself

    const bool val1 = i0 + 1 < Z;                             // the slot's second variable exists (else: computed on the
    const int i1 = val1 ? i0 + 1 : i0;                        // first one's data, nothing of it is stored)
    const unsigned line_v[V] = {(unsigned)(ca * Z + i0), (unsigned)(ca * Z + i1)};
    // the variables' own values: loaded here, first used after the edges (no load of the edge loop waits for them)
    unsigned hin[V];
    float Q[V];
#pragma unroll
    for (int v = 0; v < V; ++v) {
        hin[v] = FINAL ? 0u : a.hard_in[(int64_t)g * a.AZ + line_v[v]];
        Q[v] = a.qc[((int64_t)g * a.AZ + line_v[v]) * kIlGroup + lane];
    }
    // parities of the reporting gen rows without the variable's own decision x: bit v of odd / even = some row of
    // variable v has odd / even parity of the others; the row fails iff its parity differs from ... x (joined below)
    unsigned odd = 0, even = 0;

    // the slot's first variable's line in a run comes from an IlRef (its own offset 128 i0 sits in the base pointers);
    // the second variable's line is the next one (the halo line where the index wraps)
    const int i0b = i0 << 7;
    const float* const qT = qP + i0 * kIlGroup;
    const float* const tT = tP + i0 * kIlGroup;
    auto at = [&](const float* base, const IlRef r) { return il_at(base, r.pre - (i0b >= r.thr ? Zb : 0)); };

    // gen edge: fold every other edge of the row (the rule is associative); bit 0 of a gen edge's state is its
    // variable's hard decision: the XOR of the raw words carries sign AND parity
    auto gen_edge = [&](int k, float (&acc)[V]) {
        const GenDesc gd = s_g[k];
        const float* const tl = at(tT, s_a[k].t);
        float tv[V], num[V], den[V];
        unsigned xa[V];
#pragma unroll
        for (int v = 0; v < V; ++v) { tv[v] = __ldg(tl + v * kIlGroup); num[v] = 0.0f; den[v] = 1.0f; xa[v] = 0u; }
        // partners in batches of kGenBatch, all loads of a batch in flight (a check of degree 7, the largest of the
        // paper's ensemble, is one round trip)
        constexpr int kGenBatch = 6;
#pragma unroll 1
        for (int jb = 0; jb < gd.np; jb += kGenBatch) {
            float pm[kGenBatch][V];
#pragma unroll
            for (int u = 0; u < kGenBatch; ++u) {
                const bool have = jb + u < gd.np;
                const float* const pl = at(qT, s_p[gd.pbeg + (have ? jb + u : 0)]);
#pragma unroll
                for (int v = 0; v < V; ++v) pm[u][v] = have ? __ldg(pl + v * kIlGroup) : 0.0f;   // +0.0: the identity
            }
#pragma unroll
            for (int u = 0; u < kGenBatch; ++u)
#pragma unroll
                for (int v = 0; v < V; ++v) {
                    const unsigned wb = __float_as_uint(pm[u][v]);
                    xa[v] ^= wb;
                    boxplus_acc(__uint_as_float(wb & 0x7ffffffeu), num[v], den[v]);
                }
        }
#pragma unroll
        for (int v = 0; v < V; ++v) {
            if (!FINAL && gd.counter && (v == 0 || val1)) {   // parity of the row at the input iteration (t = (-1)^{s_c} 0)
                const unsigned par = (xa[v] ^ (__float_as_uint(tv[v]) >> 31)) & 1u;
                odd |= par << v;
                even |= (par ^ 1u) << v;
            }
            boxplus_acc(fabsf(tv[v]), num[v], den[v]);
            const float mk = with_sign(mag_of(num[v], den[v]), (xa[v] ^ __float_as_uint(tv[v])) & 0x80000000u);
            if constexpr (AS > 0) num[v] = mk;
            else mm[v * vstride + k * kstride] = mk;
            acc[v] += mk;
        }
        if constexpr (AS > 0) il_tmem_st2(tm_warp + tm_col(k), num[0], num[1]);
    };
    // edges of triple rows: two partners and an absorbed variable, one fraction, no reciprocal in between
    auto triple = [&](auto CHc, int k0, float (&acc)[V]) {
        constexpr int CH = decltype(CHc)::value;
        float tv[CH][V], pa[CH][V], pb[CH][V];
#pragma unroll
        for (int j = 0; j < CH; ++j) {
            const IlEdgeA d = s_a[k0 + j];
            const float* const tl = at(tT, d.t);
            const float* const al = at(qT, d.p);
            const float* const bl = at(qT, s_b[k0 + j].p2);
#pragma unroll
            for (int v = 0; v < V; ++v) {
                tv[j][v] = __ldg(tl + v * kIlGroup);
                pa[j][v] = __ldg(al + v * kIlGroup);
                pb[j][v] = __ldg(bl + v * kIlGroup);
            }
        }
#pragma unroll
        for (int j = 0; j < CH; ++j)
#pragma unroll
            for (int v = 0; v < V; ++v) {
                const unsigned ua = __float_as_uint(pa[j][v]), ub = __float_as_uint(pb[j][v]);
                const float qa = __uint_as_float(ua & 0x7ffffffeu), qb = __uint_as_float(ub & 0x7ffffffeu);   // bit 0: tag
                float num = qa + qb, den = fmaf(qa, qb, 1.0f);
                boxplus_acc(fabsf(tv[j][v]), num, den);
                const float mk = with_sign(mag_of(num, den), (ua ^ ub ^ __float_as_uint(tv[j][v])) & 0x80000000u);
                mm[v * vstride + (k0 + j) * kstride] = mk;
                acc[v] += mk;
            }
    };
    // pair edges: one partner and an absorbed variable
    auto pair = [&](auto CHc, int k0, float (&acc)[V]) {
        constexpr int CH = decltype(CHc)::value;
        float tv[CH][V], wv[CH][V];
#pragma unroll
        for (int j = 0; j < CH; ++j) {
            const IlEdgeA d = s_a[k0 + j];
            const float* const tl = at(tT, d.t);
            const float* const pl = at(qT, d.p);
#pragma unroll
            for (int v = 0; v < V; ++v) {
                tv[j][v] = __ldg(tl + v * kIlGroup);
                wv[j][v] = __ldg(pl + v * kIlGroup);
            }
        }
#pragma unroll
        for (int j = 0; j < CH; ++j)
#pragma unroll
            for (int v = 0; v < V; ++v) {
                const float mk = cn_rule(wv[j][v], tv[j][v]);
                mm[v * vstride + (k0 + j) * kstride] = mk;
                acc[v] += mk;
            }
    };
    using I1 = std::integral_constant<int, 1>;
    using I4 = std::integral_constant<int, 4>;
    using I8 = std::integral_constant<int, 8>;
    // block kb .. ke of this warp's partial sum `gi`: class-pure segments (gen, triple, pair), the largest chunks first
    auto block_of = [&](int rnd, int gi, int& kb, int& ke) {
        const int grp = h * GPW + gi;
        kb = (rnd * G + ((rnd & 1) ? G - 1 - grp : grp)) * kIlChunk;
        ke = min(kb + kIlChunk, dv);
    };
    float part[GPW][V];
#pragma unroll
    for (int gi = 0; gi < GPW; ++gi)
#pragma unroll
        for (int v = 0; v < V; ++v) part[gi][v] = 0.0f;
    if constexpr (AS > 0) {
        // ---- asynchronous pipeline.  Chunk c of this warp = edges k0 .. k0 + 3 of its block c / 2 (blocks in the order
        // (rnd, gi) as below), k0 = block start + 4 (c % 2); edges outside [ngh, dv) are skipped: gen edges of other gen
        // rows (k < ngh) keep their register loads (gen_edge), in order, while the copies of later chunks are in flight.
        static_assert(H == 2 && GPW == 2 && !FINAL, "built for two warps per slot; FINAL reads a buffer per lane");
        constexpr int CE = kIlAsEdges, kPer = kIlChunk / CE;  // edges per chunk, chunks per block
        unsigned char* const ring = reinterpret_cast<unsigned char*>(s_flag) + 128 + (size_t)warp * kRingWarp;   // this warp's: AS chunks x CE edges x (t | p | p2)
        const unsigned ring_s = (unsigned)__cvta_generic_to_shared(ring);
        const int half = lane >> 4;
        const unsigned l16 = (unsigned)(lane & 15) * 16u;
        const char* const qB = reinterpret_cast<const char*>(qT - lane) + l16;      // lane-free bases + this lane's 16 bytes
        const char* const tB = reinterpret_cast<const char*>(tT - lane) + l16;
        const char* const hB = half ? qB : tB;                // lanes 0-15 copy the t pair, lanes 16-31 the partner pair
        const int n_chunks = ((dv + G * kIlChunk - 1) / (G * kIlChunk)) * GPW * kPer;
        auto off_of = [&](const int pre, const int thr) { return pre - (i0b >= thr ? Zb : 0); };
        auto cp16 = [&](unsigned dst_s, const char* base, int off) {   // (base + off as ONE 32 x 32 + 64 multiply-add)
            unsigned long long src;
            asm("mad.wide.s32 %0, %1, 1, %2;" : "=l"(src) : "r"(off), "l"(reinterpret_cast<unsigned long long>(base)));
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst_s), "l"(src) : "memory");
        };
        auto issue = [&](int c) {
            if (c < n_chunks) {
                const int blk = c / kPer, rnd = blk / GPW, grp = h * GPW + (blk - rnd * GPW);
                const int k0 = (rnd * G + ((rnd & 1) ? G - 1 - grp : grp)) * kIlChunk + (c - blk * kPer) * CE;
                const unsigned e_s = ring_s + (unsigned)(c % AS) * (CE * kIlAsEdgeBytes) + l16;
                const bool whole = k0 >= ngh && k0 + CE <= dv;
#pragma unroll
                for (int j = 0; j < CE; ++j) {
                    const int k = k0 + j;
                    if (whole || (k >= ngh && k < dv)) {
                        const IlRef r = reinterpret_cast<const IlRef*>(s_a + k)[half];   // lanes 0-15: t, lanes 16-31: p
                        cp16(e_s + j * kIlAsEdgeBytes + half * 256, hB, off_of(r.pre, r.thr));
                    }
                }
                if (k0 < ng) {                                // second partners: lanes 0-15 edge 2u, lanes 16-31 edge 2u + 1
#pragma unroll
                    for (int u = 0; u < CE / 2; ++u) {
                        const int k2 = k0 + 2 * u + half;
                        if (k2 >= ngh && k2 < ng) {
                            const IlRef r = s_b[k2].p2;
                            cp16(e_s + (2 * u + half) * kIlAsEdgeBytes + 512, qB, off_of(r.pre, r.thr));
                        }
                    }
                }
            }
            il_cp_async_commit();
        };
#pragma unroll 1
        for (int c = 0; c < AS; ++c) issue(c);
        // one rolled loop over the warp's chunks (the body is large; unrolled, the kernel outgrows the instruction caches)
#pragma unroll 1
        for (int blk = 0; blk * kPer < n_chunks; ++blk) {
            const int rnd = blk / GPW, gi = blk - rnd * GPW;
            int kb, ke;
            block_of(rnd, gi, kb, ke);
            float acc[V];
#pragma unroll
            for (int v = 0; v < V; ++v) acc[v] = gi ? part[1][v] : part[0][v];
#pragma unroll 1
            for (int k = kb; k < min(ke, ngh); ++k) gen_edge(k, acc);
#pragma unroll
            for (int r2 = 0; r2 < kPer; ++r2) {
            const int c = blk * kPer + r2, k0 = kb + r2 * CE;
            il_cp_async_wait<AS - 1>();               // this thread's copies of chunk c have landed ...
            __syncwarp();                             // ... and so have the other lanes'
            const float* const e = reinterpret_cast<const float*>(ring + (size_t)(c % AS) * CE * kIlAsEdgeBytes) + lane;
            constexpr int kE = kIlAsEdgeBytes / 4;    // floats per edge of a ring entry: t at 0, p at 64, p2 at 128
            float mk[CE * V];
            if (k0 >= ng && k0 + CE <= dv) {          // pair edges only
#pragma unroll
                for (int j = 0; j < CE; ++j)
#pragma unroll
                    for (int v = 0; v < V; ++v) {
                        mk[j * V + v] = cn_rule(e[j * kE + 64 + v * kIlGroup], e[j * kE + v * kIlGroup]);
                        acc[v] += mk[j * V + v];
                    }
                il_tmem_st8(tm_warp + (unsigned)(c * CE * V), mk);
            } else if (k0 >= ngh && k0 + CE <= ng) {  // edges of triple rows only
#pragma unroll
                for (int j = 0; j < CE; ++j)
#pragma unroll
                    for (int v = 0; v < V; ++v) {
                        const float tv = e[j * kE + v * kIlGroup];
                        const unsigned ua = __float_as_uint(e[j * kE + 64 + v * kIlGroup]);
                        const unsigned ub = __float_as_uint(e[j * kE + 128 + v * kIlGroup]);
                        const float qa = __uint_as_float(ua & 0x7ffffffeu), qb = __uint_as_float(ub & 0x7ffffffeu);   // bit 0: tag
                        float num = qa + qb, den = fmaf(qa, qb, 1.0f);
                        boxplus_acc(fabsf(tv), num, den);
                        mk[j * V + v] = with_sign(mag_of(num, den), (ua ^ ub ^ __float_as_uint(tv)) & 0x80000000u);
                        acc[v] += mk[j * V + v];
                    }
                il_tmem_st8(tm_warp + (unsigned)(c * CE * V), mk);
            } else if (k0 + CE > ngh && k0 < dv) {
#pragma unroll
                for (int j = 0; j < CE; ++j) {
                    const int k = k0 + j;
                    const bool have = k >= ngh && k < dv;
                    const bool tri = k < ng;
                    const unsigned msk = tri ? 0x7ffffffeu : 0x7fffffffu;   // partners of a triple row carry a tag in bit 0
#pragma unroll
                    for (int v = 0; v < V; ++v) {
                        mk[j * V + v] = 0.0f;
                        if (have) {
                            const float tv = e[j * kE + v * kIlGroup];
                            const unsigned ua = __float_as_uint(e[j * kE + 64 + v * kIlGroup]);
                            const unsigned ub = tri ? __float_as_uint(e[j * kE + 128 + v * kIlGroup]) : 0u;
                            const float qa = __uint_as_float(ua & msk), qb = __uint_as_float(ub & msk);
                            float num = qa + qb, den = fmaf(qa, qb, 1.0f);   // (+0.0 is the identity: a pair edge)
                            boxplus_acc(fabsf(tv), num, den);
                            mk[j * V + v] = with_sign(mag_of(num, den), (ua ^ ub ^ __float_as_uint(tv)) & 0x80000000u);
                            acc[v] += mk[j * V + v];
                        }
                    }
                }
                // (the chunk may hold gen edges, whose messages gen_edge has stored: write only the others)
#pragma unroll
                for (int j = 0; j < CE; ++j)
                    if (k0 + j >= ngh && k0 + j < dv)
                        il_tmem_st2(tm_warp + (unsigned)((c * CE + j) * V), mk[j * V], mk[j * V + 1]);
            }
            __syncwarp();                             // every lane has read the ring entry: refill it
            issue(c + AS);
            }
#pragma unroll
            for (int v = 0; v < V; ++v) {
                if (gi) part[1][v] = acc[v];
                else part[0][v] = acc[v];
            }
        }
        il_cp_async_wait<0>();
    } else {
#pragma unroll 1
    for (int rnd = 0; rnd * G * kIlChunk < dv; ++rnd) {
#pragma unroll
        for (int gi = 0; gi < GPW; ++gi) {
            int k, ke;
            block_of(rnd, gi, k, ke);
            float acc[V];
#pragma unroll
            for (int v = 0; v < V; ++v) acc[v] = part[gi][v];
            const int e1 = min(ke, ngh), e3 = min(ke, ng);
            for (; k < e1; ++k) gen_edge(k, acc);
            if (MAXT <= 320) {
                if (k + 8 <= e3) { triple(I8{}, k, acc); k += 8; }
            } else {
                if (k + 4 <= e3) { triple(I4{}, k, acc); k += 4; }
            }
            if (k + 4 <= e3) { triple(I4{}, k, acc); k += 4; }
            for (; k < e3; ++k) triple(I1{}, k, acc);
            if (k + 8 <= ke) { pair(I8{}, k, acc); k += 8; }
            if (k + 4 <= ke) { pair(I4{}, k, acc); k += 4; }
            for (; k < ke; ++k) pair(I1{}, k, acc);
#pragma unroll
            for (int v = 0; v < V; ++v) part[gi][v] = acc[v];
        }
    }
    }

    // variable-node rule: the partial sums meet in the order 0 .. G-1
    float sum[V];
    if (H == 1) {
#pragma unroll
        for (int v = 0; v < V; ++v) {
            sum[v] = part[0][v];
            if (GPW > 1) {
                sum[v] = 0.0f;
#pragma unroll
                for (int gi = 0; gi < GPW; ++gi) sum[v] += part[gi][v];
            }
        }
    } else {
#pragma unroll
        for (int gi = 0; gi < GPW; ++gi)
#pragma unroll
            for (int v = 0; v < V; ++v) *xch_at(h * GPW + gi, v) = part[gi][v];
        // the two warps of this slot meet here: release / acquire on a counter in shared memory (a named barrier per
        // slot would pin all 16 hardware barriers of the CTA)
        __syncwarp();
        if (lane == 0) asm volatile("st.release.cta.s32 [%0], %1;" ::"l"(s_flag + slot * 2 + h), "r"(1) : "memory");
        int seen;
        for (;;) {
            asm volatile("ld.acquire.cta.s32 %0, [%1];" : "=r"(seen) : "l"(s_flag + slot * 2 + (1 - h)) : "memory");
            if (seen >= 1) break;
            __nanosleep(AS > 0 ? 200 : 40);                   // leave the issue slots to the others
        }
#pragma unroll
        for (int v = 0; v < V; ++v) {
            sum[v] = 0.0f;
#pragma unroll
            for (int gg = 0; gg < G; ++gg) sum[v] += *xch_at(gg, v);
        }
    }
    float L[V];
    unsigned xh[V];
#pragma unroll
    for (int v = 0; v < V; ++v) {
        L[v] = Q[v] + sum[v];                                 // L'_v
        xh[v] = __float_as_uint(L[v]) >> 31;                  // 0 iff L_v >= 0
    }
    if (FINAL) {
        if (h != 0) return;
#pragma unroll
        for (int v = 0; v < V; ++v) {
            if (live) {
                if (v == 0 || val1) {
                    const int64_t vv = (int64_t)f * a.n + (int64_t)cd.col * Z + (v ? i1 : i0);
                    a.d_hard[vv] = (uint8_t)xh[v];
                    if (a.d_post) a.d_post[vv] = L[v] * kLn2;
                }
            } else {
                xh[v] = (a.hardm[0][(int64_t)g * a.AZ + line_v[v]] >> lane) & 1u;   // t = 0: decisions of the channel values
            }
            const unsigned mask = __ballot_sync(0xffffffffu, xh[v] != 0);
            if (lane == 0 && (v == 0 || val1)) a.hardm_final[(int64_t)g * a.AZ + line_v[v]] = mask;
        }
        return;
    }
    if (h == 0) {
#pragma unroll
        for (int v = 0; v < V; ++v) {
            const unsigned mask = __ballot_sync(0xffffffffu, xh[v] != 0);
            if (lane == 0 && (v == 0 || val1)) a.hard_out[(int64_t)g * a.AZ + line_v[v]] = mask;
        }
    }
    if (ng > 0 && live) {                                     // a reporting row fails iff (parity of the others) ^ x = 1
        unsigned bad = 0;
#pragma unroll
        for (int v = 0; v < V; ++v) bad |= ((hin[v] >> lane) & 1u) ? (even >> v) & 1u : (odd >> v) & 1u;
        if (bad) a.topbad[f] = 1;
    }

    // every warp stores the new state of its own edges: w(L_vc), L_vc = L_v - m_cv = Q + sum_{k' != k} m_k'; nothing of a
    // stopped frame is stored.  The slot that holds a run's line 0 also writes the run's halo line (second round).
    if constexpr (AS > 0) asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    float* const sp0 = a.q_out + ((int64_t)g * a.EZ + (int64_t)cd.ebeg * a.Zp + i0) * kIlGroup + lane;
#pragma unroll 1
    for (int round = 0; round < (i0 == 0 ? 2 : 1); ++round) {
        float* const sp = round ? sp0 + (int64_t)Z * kIlGroup : sp0;
        const bool st[V] = {live, live && val1 && round == 0};
#pragma unroll 1
        for (int rnd = 0; rnd * G * kIlChunk < dv; ++rnd) {
#pragma unroll(AS > 0 ? 1 : GPW)
            for (int gi = 0; gi < GPW; ++gi) {
                int k, ke;
                block_of(rnd, gi, k, ke);
                float* pk = byte_ptr(sp, (unsigned)k * step);          // edge k, the slot's first variable
                if constexpr (AS > 0) {                       // the block's 16 messages come from tensor memory at once
                    if (k >= ke) continue;
                    float m16[kIlChunk * V];
                    il_tmem_ld16(tm_warp + (unsigned)((rnd * GPW + gi) * kIlChunk * V), m16);
                    if (ke - k == kIlChunk && (k >= ng || k + kIlChunk <= ng)) {   // a whole block, all of its edges with or
                        const unsigned keep = k >= ng ? 0xffffffffu : 0xfffffffeu;   // all without the tag in bit 0
#pragma unroll
                        for (int j = 0; j < kIlChunk; ++j) {
#pragma unroll
                            for (int v = 0; v < V; ++v) {
                                const unsigned wb = __float_as_uint(w_of(L[v] - m16[j * V + v]));
                                if (st[v]) il_stg(pk + v * kIlGroup, (wb & keep) | (xh[v] & ~keep));
                            }
                            pk = byte_ptr(pk, step);
                        }
                        continue;
                    }
#pragma unroll
                    for (int j = 0; j < kIlChunk; ++j) {
                        if (k + j < ke) {
                            const unsigned tagbit = (k + j < ng) ? 1u : 0u;   // gen edge: bit 0 carries the hard decision
#pragma unroll
                            for (int v = 0; v < V; ++v) {
                                const unsigned wb = __float_as_uint(w_of(single ? Q[v] : L[v] - m16[j * V + v]));
                                if (st[v]) il_stg(pk + v * kIlGroup, (wb & ~tagbit) | (xh[v] & tagbit));
                            }
                            pk = byte_ptr(pk, step);
                        }
                    }
                    continue;
                }
                const float* mk = mm + k * kstride;
                if (ke - k == kIlChunk && k >= ng) {          // a whole block without gen edges (no tag): unrolled
#pragma unroll
                    for (int j = 0; j < kIlChunk; ++j) {
#pragma unroll
                        for (int v = 0; v < V; ++v) {
                            const float wv = w_of(L[v] - mk[v * vstride + j * kstride]);
                            if (st[v]) il_stg(pk + v * kIlGroup, __float_as_uint(wv));
                        }
                        pk = byte_ptr(pk, step);
                    }
                } else {
                    for (; k < ke; ++k) {
                        const unsigned tagbit = (k < ng) ? 1u : 0u;   // gen edge: bit 0 carries the hard decision
#pragma unroll
                        for (int v = 0; v < V; ++v) {
                            const unsigned wb = __float_as_uint(w_of(single ? Q[v] : L[v] - mk[v * vstride]));
                            if (st[v]) il_stg(pk + v * kIlGroup, (wb & ~tagbit) | (xh[v] & tagbit));
                        }
                        pk = byte_ptr(pk, step);
                        mk += kstride;
                    }
                }
            }
        }
    }
    tmem_release();
}

// ---- a4: every check of every frame on the frame's frozen state (iteration d_iters[f]) -------------------------------
// Tile = 32 checks of one base row x 32 frames.  Phase 1 (lane = check): frame-major loads of the absorbed variable's
// LLR and the syndrome bit; phase 2 (lane = frame): the parity, the absorbed variable's decision (L_j = Q_j + m_cj,
// P:330); phase 3 (lane = check): frame-major stores of that variable's outputs.
__global__ void __launch_bounds__(256) k_il_check_final(const CheckTables tab, const IlArgs a) {
    __shared__ float s_q[kIlGroup][33];
    __shared__ float s_post[kIlGroup][33];
    __shared__ unsigned char s_syn[kIlGroup][36];
    __shared__ unsigned char s_xj[kIlGroup][36];
    __shared__ int s_bad[8][kIlGroup];
    const int g = blockIdx.y, lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int Z = a.Z;
    const int tiles32 = (Z + 31) / 32;
    const int R = blockIdx.x / tiles32, r0 = (blockIdx.x - R * tiles32) * 32;
    const RowDesc rd = tab.row[R];
    for (int fl = w; fl < kIlGroup; fl += 8) {
        const int f = g * kIlGroup + fl, r = r0 + lane;
        float Qj = 0.0f;
        unsigned s = 0;
        if (f < a.n_frames && r < Z) {
            if (rd.abs_col >= 0)
                Qj = __ldg(a.llr + (int64_t)f * a.n + (int64_t)rd.abs_col * Z + il_wrap(r + rd.abs_shift, Z));
            s = a.syn[(int64_t)f * a.m + (int64_t)R * Z + r] & 1u;
        }
        s_q[fl][lane] = Qj;
        s_syn[fl][lane] = (unsigned char)s;
    }
    __syncthreads();
    {
        const int f = g * kIlGroup + lane;
        const bool in_range = f < a.n_frames;
        const int T = a.iters[in_range ? f : a.n_frames - 1];
        const float* __restrict__ qprev = il_pick(a.qb, ((T > 0 ? T : 1) + 3) % 4) + (int64_t)g * a.EZ * kIlGroup;   // w^(T-1)
        const unsigned* __restrict__ hm = a.hardm_final + (int64_t)g * a.AZ;
        int nbad = 0;
        for (int rl = w; rl < 32; rl += 8) {
            const int r = r0 + rl;
            if (r >= Z) break;
            unsigned par = s_syn[lane][rl];
            unsigned sg = par << 31;
            float num = 0.0f, den = 1.0f;
#pragma unroll 4
            for (int k = 0; k < rd.ne; ++k) {
                const RowEdge re = tab.redge[rd.ebeg + k];
                const int iv = il_wrap(r + re.shift, Z);
                par ^= (hm[re.ca * Z + iv] >> lane) & 1u;
                if (rd.abs_col >= 0) {
                    unsigned wb = __float_as_uint(__ldg(il_line(qprev, (unsigned)(re.edge * a.Zp + iv), (unsigned)lane)));
                    sg ^= wb & 0x80000000u;
                    wb &= rd.gen ? 0x7ffffffeu : 0x7fffffffu;         // gen edges carry a tag in bit 0
                    boxplus_acc(__uint_as_float(wb), num, den);
                }
            }
            if (rd.abs_col >= 0) {
                const float Qj = s_q[lane][rl];
                float Lj = llr_to_log2(Qj);
                if (T > 0) Lj += with_sign(mag_of(num, den), sg);       // L'_j = Q'_j + m'_cj
                const unsigned xj = __float_as_uint(Lj) >> 31;
                s_xj[lane][rl] = (unsigned char)xj;
                s_post[lane][rl] = T > 0 ? Lj * kLn2 : Qj;
                par ^= xj;
            }
            nbad += in_range ? (int)par : 0;
        }
        s_bad[w][lane] = nbad;
    }
    __syncthreads();
    if (w == 0) {                                             // one atomic per frame and CTA (thousands of CTAs, 32 addresses)
        int nbad = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) nbad += s_bad[k][lane];
        if (nbad) atomicAdd(a.unsat + g * kIlGroup + lane, nbad);
    }
    if (rd.abs_col < 0) return;                               // block-uniform
    for (int fl = w; fl < kIlGroup; fl += 8) {
        const int f = g * kIlGroup + fl, r = r0 + lane;
        if (f < a.n_frames && r < Z) {
            const int64_t v = (int64_t)f * a.n + (int64_t)rd.abs_col * Z + il_wrap(r + rd.abs_shift, Z);
            a.d_hard[v] = s_xj[fl][lane];
            if (a.d_post) a.d_post[v] = s_post[fl][lane];
        }
    }
}
#endif

// ---- host side --------------------------------------------------------------------------------------------------------
struct IlLaunch {
    PassTables tab; CheckTables ctab; IlArgs args; cudaStream_t stream;
    const CheckArgs* check;    // the early-exit check this launch carries in its grid (NULL: none)
    bool final_mode; int n_sm, prepare_only;
};

// variables per CTA (an even number: slots of two): H warps per slot; long columns (H = 2) take five slots -- the
// 320-thread instance, two CTAs of 10 warps per multiprocessor --, short ones up to twelve; never more slots than a
// column has, and two CTAs per multiprocessor must fit the shared memory
inline int il_pick_w(int Z, int max_dv, int max_np) {
    const int H = max_dv > 2 * kIlChunk ? 2 : 1, spc = (Z + 1) / 2;
    int sl = std::min(spc, H == 2 ? 5 : 12);
    while (sl > 1 && il_smem_bytes(max_dv, max_np, 2 * sl) > 110 * 1024) --sl;
    return 2 * sl;
}

#ifdef QC_IL_IMPL
template <int H, int GPW, int MAXT, int AS>
inline void launch_pass_il_h(const IlLaunch& L) {
    IlArgs args = L.args;
    const int threads = 32 * H * (args.W / 2);
    const size_t smem = il_smem_bytes(args.max_dv, args.max_np, args.W, AS, threads / 32);
    static thread_local int attr_dev = -1;                  // the attribute is per device
    int dev = 0;
    cudaGetDevice(&dev);
    if (attr_dev != dev) {
        cudaFuncSetAttribute(k_pass_il<true, H, GPW, MAXT, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 208 * 1024);
        cudaFuncSetAttribute(k_pass_il<false, H, GPW, MAXT, AS>, cudaFuncAttributeMaxDynamicSharedMemorySize, 208 * 1024);
        attr_dev = dev;
    }
    if (L.prepare_only) return;
    const bool with_check = !L.final_mode && L.check != nullptr;
    const int work = (args.n_cols * args.spc + args.ipc - 1) / args.ipc;
    const int extra = with_check ? (2 * L.n_sm + args.n_groups - 1) / args.n_groups : 0;
    args.cand_x = with_check ? work : -1;
    static const CheckTables no_tab{nullptr, nullptr};
    static const CheckArgs no_args{};
    const dim3 grid(work + extra, args.n_groups), block(threads);
    if (L.final_mode)
        k_pass_il<true, H, GPW, MAXT, 0><<<grid, block, il_smem_bytes(args.max_dv, args.max_np, args.W), L.stream>>>(
            L.tab, args, no_tab, no_args);                  // (FINAL reads a buffer per lane: register loads)
    else
        launch_pdl(k_pass_il<false, H, GPW, MAXT, AS>, grid, block, smem, L.stream, L.tab, args, with_check ? L.ctab : no_tab,
                   with_check ? *L.check : no_args);
}

// long columns (four partial sums): two warps per variable; short ones: one warp, one sum
inline void launch_pass_il(const IlLaunch& L) {
    if (L.args.split == 4) {
        const bool narrow = 32 * 2 * (L.args.W / 2) <= 320;
        if (L.args.as_depth > 0 && 32 * 2 * (L.args.W / 2) <= 256) {   // four CTAs per multiprocessor
            switch (L.args.as_depth) {
                case 1: launch_pass_il_h<2, 2, 256, 1>(L); break;
                case 2: launch_pass_il_h<2, 2, 256, 2>(L); break;
                case 3: launch_pass_il_h<2, 2, 256, 3>(L); break;
                default: launch_pass_il_h<2, 2, 256, 4>(L); break;
            }
            return;
        }
        switch (narrow ? L.args.as_depth : 0) {
            case 1: launch_pass_il_h<2, 2, 320, 1>(L); break;
            case 2: launch_pass_il_h<2, 2, 320, 2>(L); break;
            case 3: launch_pass_il_h<2, 2, 320, 3>(L); break;
            case 4: launch_pass_il_h<2, 2, 320, 4>(L); break;
            default:
                if (narrow) launch_pass_il_h<2, 2, 320, 0>(L);
                else launch_pass_il_h<2, 2, 384, 0>(L);
        }
    } else {
        launch_pass_il_h<1, 1, 384, 0>(L);
    }
}
#endif

}  // namespace qc

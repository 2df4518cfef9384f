// Shared declarations of libqcldpc's translation units (tables, kernel arguments, device helpers).
// Citations "P:NNN" are /root/reference/PAPER.md lines; readings S1.. are listed in DESIGN.md.
#pragma once

#include <cuda_runtime.h>

#include <cstdint>

#include "../../include/qcldpc.h"
#include "../../include/qcldpc_profile.h"

namespace qc {

constexpr int kMaxDv = 64;          // largest supported active-column degree
constexpr int kThreads = 128;       // threads per CTA in every kernel
constexpr int kMaxV = 2;            // variables per thread in k_pass (tile = kThreads * V consecutive variables)
constexpr int kHalo = kThreads * kMaxV;   // every cyclic run of Z floats is stored with this many wrapped copies behind it
constexpr int kMaxPartners = 2048;  // partner entries (other edges of the gen rows) per active column
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
constexpr float kMsgMax2 = QCLDPC_MSG_MAX * kLog2e;   // the clamp S2 in log2 units

// ---- layout -----------------------------------------------------------------------------------------------------
// Messages live in base-2 units: L' = L * log2(e).  Edge state of active edge e = (c,v), variable index i:
//     w[e * Zs + i] = sgn(L_vc) * 2^-|L'_vc|          (sign in the IEEE sign bit; S3: -0 never occurs)
// Zs = round_up(Z + kHalo, 32): the run [0,Z) is followed by a copy of its first kHalo entries, so that a tile of
// consecutive variables reads its cyclically shifted window [a, a + tile) with a < Z WITHOUT a per-element wrap.
// (Codes of the generic pass: compact runs, Zs = round_up(Z, 8), no halo, the reader wraps per element.)
// Edges of "gen" rows (see below) carry the hard decision xhat_v of their variable in mantissa bit 0 (the reader
// masks it off: the magnitude never depends on it).
// Static per check c of base row R, index r:
//     t[R * Zs + r] = (-1)^{s_c} * sgn(Q_j) * 2^-|Q'_j|   for the absorbed degree-1 variable j of c, or
//                     (-1)^{s_c} * 0                       if the row has none                   (same halo).

// ---- code tables (built once by qcldpc_code_create, read from global memory in each block's preamble) -----------
// A base row is a PAIR row if it has an absorbed variable and exactly two active edges (every lower row of the
// BASELINE.json codes); every other row is a GEN row.  Inside an active column the gen edges come first.
// A TRIPLE row is a gen row with an absorbed variable and exactly three active edges (the lower rows of the paper's
// ensemble): its edges have two partners and no parity to report; the generic pass gives them a predicate-free body.
struct EdgeDesc {                       // t at t[t_off + (i - shift) mod Z]
    int shift; int t_off;
    int p_off; int delta;               // pair or triple edge: partner at w[p_off + (i + delta) mod Z], else p_off = -1
    int p2_off; int delta2;             // triple edge: second partner, else p2_off = -1
};
struct GenDesc { int pbeg; int np; int counter; int pad; };       // partners [pbeg, pbeg+np) relative to the column's
                                                                  // first partner; counter: this edge reports the row's parity
struct PartnerDesc { int off; int delta; };                       // w[off + (i + delta) mod Z]
struct ColDesc { int col; int ebeg; int dv; int ng; int gbeg; int pbeg; int np; int ngh; };
// edges of a column: [0, ngh) gen edges of other gen rows, [ngh, ng) gen edges of triple rows, [ng, dv) pair edges
struct RowDesc { int ebeg; int ne; int abs_col; int abs_shift; int gen; int pad0, pad1, pad2; };   // gen: 0 pair, 1 gen, 2 triple
struct RowEdge { int edge; int shift; int col; int ca; };         // active edge seen from its row (ca = active column)

struct PassTables { const EdgeDesc* edge; const GenDesc* gen; const PartnerDesc* partner; const ColDesc* col; };
struct CheckTables { const RowDesc* row; const RowEdge* redge; };

// ---- kernel arguments -------------------------------------------------------------------------------------------
struct PassArgs {
    const float* llr;          // [F][n]
    float* qb[4];              // the four edge-state buffers [F][E][Zs] (iteration t lives in buffer t mod 4: check.cuh)
    const float* t;            // [F][mb][Zs]
    const uint8_t* hard_in;    // xhat of the input iteration, active columns only [F][A][Zs]
    uint8_t* hard_out;
    uint8_t* d_hard;           // FINAL: outputs
    float* d_post;
    const int* done;           // [F]
    const int32_t* iters;      // [F]  (FINAL: the iteration whose decisions are formed)
    int* topbad;               // [F]  slot of the input iteration: set to 1 if a parity of a row without absorbed variable fails
    int in_buf, out_buf;       // regular pass: qb[in_buf] -> qb[out_buf]
    int Z, Zs, tiles;
    int table_bytes, max_dv;   // generic kernel: bytes of its shared-memory tables; messages [max_dv][FV][TB] follow
    int n_frames;              // generic kernel: frames of the batch (two per thread when batched)
    int cand_y;                // exact kernels: blockIdx.y of the CTAs that run the early-exit check (check.cuh), or -1
    int64_t n, EZs, mZs, AZs;  // per-frame strides
    int pack;                  // generic pass: frames side by side in one tile (circulants of at most half a tile), >= 1
    int flip;                  // 1: the grid walks the frames backwards (odd iterations: the frames the previous launch
                               // wrote last, still in L2, are read first)
};

// Codes whose active columns all have the same shape (DV edges, the first NG of them gen edges; at most kMaxExactCols
// columns): the column descriptors travel in the kernel parameters (pass_exact.cuh).  Offsets are in floats.
constexpr int kMaxExactCols = 16;
template <int DV, int NG, int PCAP>
struct ExactCol {
    int col, ebeg;                                   // base column; first active edge
    int shift[DV], t_off[DV];                        // edge k: t at t[t_off + (i - shift) mod Z]
    int p_off[DV], delta[DV];                        // pair edge k >= NG: partner at w[p_off + (i + delta) mod Z]
    int g_off[(NG > 0 ? NG : 1) * PCAP], g_delta[(NG > 0 ? NG : 1) * PCAP];   // gen edge g, slot j: partner or off = -1
    int g_np[NG > 0 ? NG : 1], g_counter[NG > 0 ? NG : 1], g_pbeg[NG > 0 ? NG : 1];   // all partners: partner[g_pbeg + j], j < g_np
};
template <int DV, int NG, int PCAP>
struct ExactTable { ExactCol<DV, NG, PCAP> c[kMaxExactCols]; };
struct HostTables { const EdgeDesc* edge; const GenDesc* gen; const PartnerDesc* partner; const ColDesc* col; int n_cols; };

struct PassLaunch {
    PassTables tab; PassArgs args; cudaStream_t stream; int V; bool final_mode;
    const void* exact;         // HOST: the ExactTable of the instantiation (exact families only)
    const void* check_tab;     // HOST: CheckTables / CheckArgs of the early-exit check this launch carries in its grid
    const void* check_args;    //       (exact families; NULL: none)
    int n_cols, n_frames, max_np, max_dv;
    int n_sm;                  // multiprocessors of the device
    int fv;                    // generic pass: frames per thread (1 or 2)
    int pack_ok;               // generic pass: lane packing allowed
    int prepare_only;          // 1: set the kernel attributes of the instantiation this launch would use, launch nothing
};
using PassLauncher = void (*)(const PassLaunch&);
using ExactBuilder = size_t (*)(const HostTables&, void* out);   // out = NULL: size only

// Programmatic dependent launch: the per-iteration kernels (the fused pass, k_cand) are launched with
// cudaLaunchAttributeProgrammaticStreamSerialization, so the CTAs of launch k+1 are placed on the SMs while launch k
// drains, run their parameter-only preamble and block in pdl_wait() until launch k has completed and its writes are
// visible.  Every such kernel calls pdl_launch() first and pdl_wait() before its first access to global memory that
// a predecessor writes -- in EVERY CTA, so completion of launch k+1 implies completion of launch k (the chain is
// transitive).
template <class... KArgs, class... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// ---- device helpers ---------------------------------------------------------------------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ float ex2_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float lg2_approx(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rcp_approx(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// LLR in base-2 units; "+ 0.0f" turns -0.0 into +0.0 so that the sign bit alone is "L < 0" from here on (S3)
__device__ __forceinline__ float llr_to_log2(float Q) { return Q * kLog2e + 0.0f; }
// w(L') = sgn(L') 2^-|L'|
__device__ __forceinline__ float w_of(float L2) {
    const float q = ex2_approx(-fabsf(L2));
    return __uint_as_float(__float_as_uint(q) | (__float_as_uint(L2) & 0x80000000u));
}
// |m'| = lg2 den - lg2 num, clamped (S2).  num = 0 -> +inf -> clamp.
__device__ __forceinline__ float mag_of(float num, float den) {
    return fminf(lg2_approx(den) - lg2_approx(num), kMsgMax2);
}
// (num/den) [+] a = (num + a den) / (den + a num): the check-node rule on q = 2^-|L'| values, fraction kept apart
__device__ __forceinline__ void boxplus_acc(float a, float& num, float& den) {
    const float n2 = fmaf(a, den, num);
    den = fmaf(a, num, den);
    num = n2;
}
// base + boff bytes as ONE 32x32+64 multiply-add (IMAD.WIDE.U32 with multiplier 1; a multiplier of 4 is split by ptxas
// into LEA + LEA.HI.X); boff is an unsigned byte offset < 2^32
template <class T>
__device__ __forceinline__ T* byte_ptr(T* base, unsigned boff) {
    unsigned long long r;
    asm("mad.wide.u32 %0, %1, 1, %2;" : "=l"(r) : "r"(boff), "l"((unsigned long long)base));
    return reinterpret_cast<T*>(r);
}
__device__ __forceinline__ unsigned sign_of(float x) { return __float_as_uint(x) & 0x80000000u; }
// XOR, not OR: the approximate lg2/rcp can make a magnitude that should be +0 come out as -tiny, and the result must
// stay an odd function of the signs (the syndrome <-> codeword equivalence is bit-exact, tests P5)
__device__ __forceinline__ float with_sign(float mag, unsigned sg) { return __uint_as_float(__float_as_uint(mag) ^ sg); }
// check-node rule of a row with one other active edge: partner [+] static term; the sign product includes
// (-1)^{s_c} via t
__device__ __forceinline__ float cn_rule(float wv, float tv) {
    const float qa = fabsf(wv), tt = fabsf(tv);
    return with_sign(mag_of(qa + tt, fmaf(qa, tt, 1.0f)), sign_of(wv) ^ sign_of(tv));
}
#endif

}  // namespace qc

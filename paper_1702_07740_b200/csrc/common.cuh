// Shared declarations of libqcldpc's translation units (tables, kernel arguments, device helpers).
// Citations "P:NNN" are /root/reference/PAPER.md lines; readings S1.. are listed in DESIGN.md.
#pragma once

#include <cuda_runtime.h>

#include <cstdint>

#include "../../include/qcldpc.h"

namespace qc {

constexpr int kMaxDv = 64;       // largest supported active-column degree
constexpr int kThreads = 128;    // threads per CTA in every kernel
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

// ---- code tables (built once by qcldpc_code_create) -----------------------------------------------------------
// Active edge seen from its own variable.  Check index r = (i - shift) mod Z; static term at t[t_off + r].
// If the row has exactly one other active edge ("pair row", every lower row of the BASELINE.json codes) that
// partner's message sits at q[p_off + (i + delta) mod Z]; otherwise p_off = -1 and a GenDesc lists the partners.
struct PairDesc { int shift; int t_off; int p_off; int delta; };
struct GenDesc { int k; int pbeg; int np; int pad; };             // k: edge index inside the column
struct PartnerDesc { int off; int delta; };                       // q[off + (i + delta) mod Z]
struct ColDesc { int col; int ebeg; int dv; int gbeg; int ng; int pad0, pad1, pad2; };
struct RowDesc { int ebeg; int ne; int abs_col; int abs_shift; }; // base row: active edges, absorbed column or -1
struct RowEdge { int edge; int shift; int col; int pad; };        // active edge seen from its row

// Tables small enough travel as __grid_constant__ kernel parameters (constant bank, uniform loads); larger codes
// read the same tables from global memory.
constexpr int kInlEdges = 256, kInlPartners = 512, kInlCols = 32, kInlGen = 96, kInlRows = 128;
struct VnTablesInline {
    PairDesc pair[kInlEdges]; PartnerDesc partner[kInlPartners]; GenDesc gen[kInlGen]; ColDesc col[kInlCols];
};
struct VnTablesGlobal { const PairDesc* pair; const PartnerDesc* partner; const GenDesc* gen; const ColDesc* col; };
struct CnTablesInline { RowDesc row[kInlRows]; RowEdge redge[kInlEdges]; };
struct CnTablesGlobal { const RowDesc* row; const RowEdge* redge; };

// ---- kernel arguments -------------------------------------------------------------------------------------------
struct VnArgs {
    const float* llr; const float* qold; float* qnew; const float* t; uint8_t* hard; float* post; const int* done;
    int Z, tiles; int64_t n, m, EZ;
};

struct VnLaunch {
    const VnTablesInline* inl;    // host pointer, or nullptr -> use `glob`
    VnTablesGlobal glob;
    VnArgs args;
    dim3 grid;
    cudaStream_t stream;
};
using VnLauncher = void (*)(const VnLaunch&);

// ---- device helpers -----------------------------------------------------------------------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ float ex2_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float lg2_approx(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// q(L) = sgn(L) exp(-|L|); sgn(x) = -1 iff x < 0, so -0.0 counts as + (reading S3)
__device__ __forceinline__ float q_of_llr(float L) {
    const float q = ex2_approx(-fabsf(L) * kLog2e);
    return __uint_as_float(__float_as_uint(q) | (L < 0.0f ? 0x80000000u : 0u));
}
// |m| = ln den - ln num, clamped (S2).  num = 0 -> +inf -> clamp.
__device__ __forceinline__ float mag_of(float num, float den) {
    return fminf(kLn2 * (lg2_approx(den) - lg2_approx(num)), QCLDPC_MSG_MAX);
}
// (num/den) [+] a = (num + a den) / (den + a num): Moebius addition of q = exp(-|L|) values, fraction kept apart
__device__ __forceinline__ void boxplus_acc(float a, float& num, float& den) {
    const float n2 = fmaf(a, den, num);
    den = fmaf(a, num, den);
    num = n2;
}
__device__ __forceinline__ unsigned sign_of(float x) { return __float_as_uint(x) & 0x80000000u; }
__device__ __forceinline__ float with_sign(float mag, unsigned sg) { return __uint_as_float(__float_as_uint(mag) | sg); }
#endif

}  // namespace qc

// libqcldpc -- B200 (sm_100a) flooding Sum-Product decoder for QC-LDPC codes in syndrome form.
// C ABI: include/qcldpc.h.  Design notes: DESIGN.md.  Citations "P:NNN" are /root/reference/PAPER.md lines.
//
// Arithmetic domain.  Edge state is stored as  w_vc = sgn(L_vc) * 2^-|L'_vc|,  L' = L log2(e)  (sign in the IEEE sign
// bit).  With tanh(|L|/2) = (1-q)/(1+q), q = e^-|L|, the paper's check-node rule
//     |m_cv| = Phi^-1( sum_{v'} Phi(|L_v'c|) ) = 2 atanh( prod_{v'} tanh(|L_v'c|/2) )
// becomes a Moebius ("velocity") addition of the q's,  q_a [+] q_b = (q_a + q_b) / (1 + q_a q_b),
// and |m_cv| = -ln( [+]_{v' in N(c)\v} q_v'c ).  Keeping numerator and denominator apart,
//     (num, den) <- (num + a*den, den + a*num),   |m'_cv| = lg2 den - lg2 num,
// needs no division, no cancellation (all terms are >= 0) and one ex2 + two lg2 per edge and iteration.
// Degree-1 variables that are absorbed into their row contribute a constant q, folded together with the
// syndrome sign (-1)^{s_c} (reading S1) into one static float per check, t_c.
//
// Kernels:
//   k_init_cols a0  w^(0) = w(Q_v) on every active edge (+ halo), decisions at t = 0 of the active variables
//   k_init_rows a0  t_c from the absorbed variable's LLR and the syndrome bit (+ halo)
//   k_pass_exact / k_pass  a1+a2  (pass_exact.cuh: the BASELINE.json column shapes, tables in kernel parameters;
//               pass_kernel.cuh: any code, the paper's own ensemble included) fused check-node + variable-node update
//               of one iteration, VN-centric; also forms, from bit-0 tags, the parity of the rows WITHOUT absorbed
//               variable at the previous iteration: a necessary condition for H xhat = s that costs no extra traffic.
//               Launched with programmatic dependent launch (common.cuh), like k_cand.
//   cand_work   a3  (check.cuh) early exit: for the frames that pass that filter, the full check (decisions of the
//               absorbed variables L_j = Q_j + m_cj and every parity) on the still intact state of that iteration;
//               returns at once when there is no candidate; freezes d_iters / d_pass / done per frame.  Runs in an
//               extra grid row of k_pass_exact, or as the stand-alone k_cand (generic family, last iteration).
//   the FINAL instantiations of the pass, k_check_final, k_flags_final   a4  outputs from each frame's frozen state
//   k_pass_il, k_il_*, k_cand_il   the same steps on the frame-interleaved layout (pass_il.cuh): batches of codes with
//               long columns, the paper's own ensemble above all
//   k_loop_ctl  the iteration loop itself: one CUDA graph per decode with a conditional WHILE node (decode_impl)
//   (the steps either side of the decoder -- LLR front end, bit packing, CRC-32 -- are in frontend.cu)
// Edge state lives in four buffers (iteration t in buffer t mod 4); the early-exit check of iteration t-2 runs next to
// pass t and touches nothing that pass writes: check.cuh has the timeline.
#include "check.cuh"
#include "common.cuh"
#include "pass_il.cuh"

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

namespace qc {
// one object file per instantiation family of k_pass (pass_inst.cu)
void launch_pass_dv11_ng3(const PassLaunch&);
void launch_pass_dv21_ng3(const PassLaunch&);
void launch_pass_generic(const PassLaunch&);
size_t launch_pass_dv11_ng3_table(const HostTables&, void*);
size_t launch_pass_dv21_ng3_table(const HostTables&, void*);
// the frame-interleaved family (pass_il.cu)
void launch_pass_il_entry(const IlLaunch&);
void launch_il_init(const PassTables&, const CheckTables&, const IlArgs&, cudaStream_t);
void launch_il_cand(const CheckTables&, const CheckArgs&, const IlArgs&, int blocks, cudaStream_t);
void launch_il_check_final(const CheckTables&, const IlArgs&, cudaStream_t);
}  // namespace qc

using namespace qc;

namespace {

thread_local char g_cuda_error[512] = "";
thread_local int64_t g_launches = 0;
thread_local int g_loop_mode = 0;         // 1: the last decode of this thread ran as a graph with a device-side loop

// Optional launch timing (qcldpc_profile_enable): CUDA event pairs around sampled launches, on the decode stream.
struct Profile {
    int stride = 0;                       // 0 = off
    std::vector<cudaEvent_t> pool;        // reused across calls
    std::vector<int> kind;                // kind of pair k (events 2k, 2k+1)
    int64_t launched[2] = {0, 0};
};
thread_local Profile g_prof;

}  // namespace

// Tuning knobs (defaults are the measured best).  Part of the immutable handle: the decode calls read no
// environment variable and keep no state outside the handle and the caller's workspace.
struct Tuning {
    int V = 0;                            // QCLDPC_V=1|2: variables per thread of k_pass_exact (0: by grid size)
    int flip = 1;                         // QCLDPC_FLIP=0: every launch walks the frames forwards
    int merge_check = 1;                  // QCLDPC_MERGE_CHECK=0: the early-exit check is a separate k_cand launch
    int cand_per_sm = 0;                  // QCLDPC_CAND_PER_SM=k: grid of a separate k_cand launch (0: by batch size)
    int pack = 1;                         // QCLDPC_PACK=0: no lane packing in the generic pass
    int fv = 0;                           // QCLDPC_FV=1|2: frames per thread of the generic pass (0: by batch size)
    int loop_graph = 1;                   // QCLDPC_LOOP=stream: one launch per iteration from the host, no graph
    int body_mult = 0;                    // QCLDPC_BODY=k: the graph loop's body is 12 k iterations (0: by batch size)
    int il = 1;                           // QCLDPC_IL=0: never the frame-interleaved family; 2: for every batch size
};

// One instantiated decode graph per argument tuple (the kernel parameters are baked into the graph's nodes).
struct GraphKey {
    const void *llr, *syn, *hard, *iters, *pass, *post, *ws;
    int n_frames, max_iter, early_stop, check_from, device;
};
struct GraphEntry { GraphKey key; cudaGraphExec_t exec; uint64_t stamp; };

static int env_int(const char* name, int dflt) {
    const char* e = getenv(name);
    return (e && *e) ? atoi(e) : dflt;
}

struct qcldpc_code {
    int mb, nb, Z, Zs, tiles;             // tiles = ceil(Z / kThreads)
    int halo = 0, max_np = 0;             // halo: runs are followed by kHalo wrapped entries (exact families)
    int64_t n, m;
    int n_act_cols, n_act_edges, max_dv;
    bool filter_rows;                     // some row has no absorbed variable (the early-exit filter exists)
    std::vector<EdgeDesc> edge;
    std::vector<GenDesc> gen;
    std::vector<PartnerDesc> partner;
    std::vector<ColDesc> col;
    std::vector<RowDesc> row;
    std::vector<RowEdge> redge;
    EdgeDesc* d_edge = nullptr; GenDesc* d_gen = nullptr; PartnerDesc* d_partner = nullptr; ColDesc* d_col = nullptr;
    RowDesc* d_row = nullptr; RowEdge* d_redge = nullptr;
    // frame-interleaved family (pass_il.cuh): the same tables with run length Z (a run is Z lines of 32 frames)
    std::vector<EdgeDesc> edge_il; std::vector<PartnerDesc> partner_il;
    EdgeDesc* d_edge_il = nullptr; PartnerDesc* d_partner_il = nullptr;
    std::vector<uint4> il_blob; uint4* d_il_blob = nullptr; int il_blob16 = 0;   // per-column tables of k_pass_il
    bool il_ok = false;                   // the code fits the family's 32-bit byte offsets
    int il_w = 8;                         // warps per CTA of k_pass_il
    int il_as = 0;                        // chunks a warp of k_pass_il keeps in flight by asynchronous copies (0: none)
    PassLauncher launcher = nullptr;
    std::vector<char> exact;              // kernel-parameter table of the exact family (empty: generic kernel)
    int n_sm = 148;
    Tuning tune;                          // read ONCE from the environment by qcldpc_code_create (include/qcldpc.h)
    // graph cache: the only mutable part of the handle, guarded by graph_mu (decode calls take a const handle)
    std::mutex graph_mu;
    std::vector<GraphEntry> graphs;
    uint64_t graph_clock = 0;
    cudaStream_t cap_main = nullptr, cap_body = nullptr;   // capture-only streams: nothing ever executes on them
};

namespace {

struct InitArgs {
    const float* llr; const uint8_t* syn; float* q0; float* t; uint8_t* hard0; uint8_t* d_hard; float* d_post;
    int Z, Zs, tiles, halo; int64_t n, m, EZs, mZs, AZs;
};

// a0: w^(0) on every active edge, decisions at t = 0 for active variables.  One thread per (active column, index).
__global__ void __launch_bounds__(kThreads) k_init_cols(const PassTables tab, const InitArgs a) {
    const int f = blockIdx.y;
    const int ca = blockIdx.x / a.tiles;
    const int i = (blockIdx.x - ca * a.tiles) * kThreads + threadIdx.x;
    if (i >= a.Z) return;
    const ColDesc cd = tab.col[ca];
    const int64_t v = (int64_t)f * a.n + (int64_t)cd.col * a.Z + i;
    const float Q = __ldg(a.llr + v);
    const float Q2 = llr_to_log2(Q);
    const unsigned xh = __float_as_uint(Q2) >> 31;
    const unsigned wb = __float_as_uint(w_of(Q2));
    float* q0 = a.q0 + (int64_t)f * a.EZs + (int64_t)cd.ebeg * a.Zs;
    const bool halo = a.halo && i < kHalo;
    for (int k = 0; k < cd.dv; ++k) {
        const float w = __uint_as_float(k < cd.ng ? ((wb & 0xfffffffeu) | xh) : wb);
        q0[(int64_t)k * a.Zs + i] = w;
        if (halo) q0[(int64_t)k * a.Zs + a.Z + i] = w;
    }
    a.hard0[(int64_t)f * a.AZs + (int64_t)ca * a.Zs + i] = (uint8_t)xh;
    a.d_hard[v] = (uint8_t)xh;
    if (a.d_post) a.d_post[v] = Q;
}

// a0: t_c = (-1)^{s_c} sgn(Q_j) 2^-|Q'_j| for the absorbed variable j of check c, or (-1)^{s_c} * 0
__global__ void __launch_bounds__(kThreads) k_init_rows(const CheckTables tab, const InitArgs a) {
    const int f = blockIdx.y;
    const int R = blockIdx.x / a.tiles;
    const int r = (blockIdx.x - R * a.tiles) * kThreads + threadIdx.x;
    if (r >= a.Z) return;
    const RowDesc rd = tab.row[R];
    const int64_t c = (int64_t)R * a.Z + r;
    float t = 0.0f;
    if (rd.abs_col >= 0) {
        int j = r + rd.abs_shift; j -= (j >= a.Z) ? a.Z : 0;
        t = w_of(llr_to_log2(__ldg(a.llr + (int64_t)f * a.n + (int64_t)rd.abs_col * a.Z + j)));
    }
    const unsigned s = a.syn[(int64_t)f * a.m + c] & 1u;
    const float ts = __uint_as_float(__float_as_uint(t) ^ (s << 31));
    float* tf = a.t + (int64_t)f * a.mZs + (int64_t)R * a.Zs;
    tf[r] = ts;
    if (a.halo && r < kHalo) tf[a.Z + r] = ts;
}

// a4: one thread per check of every frame, on the frame's frozen state (iteration d_iters[f]); counts failed parities
__global__ void __launch_bounds__(kThreads) k_check_final(const CheckTables tab, const CheckArgs a) {
    const int f = blockIdx.y;
    const int R = blockIdx.x / a.tiles;
    const int r = (blockIdx.x - R * a.tiles) * kThreads + threadIdx.x;
    unsigned bad = 0;
    if (r < a.Z) bad = check_one<true>(tab, a, f, R, r, a.iters[f]);
    const int nbad = __syncthreads_count(bad != 0);
    if (threadIdx.x == 0 && nbad) atomicAdd(a.unsat + f, nbad);
}

__global__ void k_flags_final(int* unsat, uint8_t* pass, int n_frames) {
    const int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= n_frames) return;
    pass[f] = unsat[f] == 0 ? 1 : 0;
    unsat[f] = 0;
}

// a3, stand-alone launch of the early-exit work (check.cuh): the generic kernel family, and the last checked iteration
// of every decode
__global__ void __launch_bounds__(kThreads) k_cand(const CheckTables tab, const CheckArgs a) {
    pdl_launch();
    pdl_wait();
    cand_work(tab, a, blockIdx.x, gridDim.x, threadIdx.x, kThreads);
}

// number of frames still iterating (decode_host polls it between chunks of iterations)
__global__ void k_live_count(const int* done, int n_frames, int* n_live) {
    int c = 0;
    for (int f = threadIdx.x; f < n_frames; f += blockDim.x) c += done[f] ? 0 : 1;
    __shared__ int s_c;
    if (threadIdx.x == 0) s_c = 0;
    __syncthreads();
    if (c) atomicAdd(&s_c, c);
    __syncthreads();
    if (threadIdx.x == 0) *n_live = s_c;
}

// Device-side state of the iteration loop: ints behind the grid ticket in the workspace.
enum LoopCtl { kCtlLive = 16,        // host-polling path: frames still iterating, read back every kPollEvery launches
               kCtlIterBase = 32,    // graph path: iterations the WHILE loop has completed (a multiple of the body length)
               kCtlNLive = 33,       // frames still iterating, as of the last early-exit check that ran (cand_work)
               kCtlStopped = 34,     // the loop ended because every frame had stopped (not because of max_iter)
               kCtlIssued = 35 };    // passes launched by the decode call (qcldpc_iterations_issued)

__global__ void k_reset(int* done2, int* unsat, int* topbad3, int* fullbad, unsigned* ticket, int32_t* iters,
                        uint8_t* pass, int n_frames, int max_iter) {
    const int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f == 0) {
        *ticket = 0;
        int* ctl = reinterpret_cast<int*>(ticket);
        ctl[kCtlIterBase] = 0; ctl[kCtlNLive] = n_frames; ctl[kCtlStopped] = 0; ctl[kCtlIssued] = 0;
    }
    if (f >= n_frames) return;
    done2[f] = 0; done2[n_frames + f] = 0; unsat[f] = 0; fullbad[f] = 0;
    topbad3[f] = 0; topbad3[n_frames + f] = 0; topbad3[2 * n_frames + f] = 0;
    iters[f] = max_iter; pass[f] = 0;
}

// End of one body of the graph WHILE loop (`body` iterations): advance the iteration base and decide whether the loop
// runs again: iterations remain AND some frame is still iterating ("Go to Step 5" for the whole batch).
__global__ void k_loop_ctl(cudaGraphConditionalHandle handle, int* ctl, int body, int loop_iters, int pre_iters) {
    const int completed = ctl[kCtlIterBase] + body;
    ctl[kCtlIterBase] = completed;
    ctl[kCtlIssued] = pre_iters + completed;
    const bool more = completed < loop_iters;
    const bool live = ctl[kCtlNLive] > 0;
    if (more && !live) ctl[kCtlStopped] = 1;
    cudaGraphSetConditional(handle, (more && live) ? 1u : 0u);
}

__global__ void k_set_int(int* p, int v) { *p = v; }

// ---------------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------------
// kind 0 = k_pass, 1 = k_cand.  Returns the pair index to close with prof_end, or -1.
int prof_begin(int kind, cudaStream_t st) {
    Profile& p = g_prof;
    if (p.stride <= 0) return -1;
    const int64_t seq = p.launched[kind]++;
    if (seq % p.stride) return -1;
    const size_t k = p.kind.size();
    while (p.pool.size() < 2 * (k + 1)) {
        cudaEvent_t ev;
        if (cudaEventCreate(&ev) != cudaSuccess) return -1;
        p.pool.push_back(ev);
    }
    p.kind.push_back(kind);
    cudaEventRecord(p.pool[2 * k], st);
    return (int)k;
}
void prof_end(int k, cudaStream_t st) {
    if (k >= 0) cudaEventRecord(g_prof.pool[2 * k + 1], st);
}

int cuda_fail(cudaError_t e, const char* what) {
    snprintf(g_cuda_error, sizeof(g_cuda_error), "%s: %s", what, cudaGetErrorString(e));
    return QCLDPC_ERR_CUDA;
}
#define CUDA_TRY(call)                                                      \
    do {                                                                    \
        cudaError_t e_ = (call);                                            \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);                 \
    } while (0)

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Workspace {
    float* qbuf[4]; float* t; uint8_t* hardbuf[3]; int* done; int* unsat; int* topbad; int* fullbad; unsigned* ticket;
    // frame-interleaved family: LLRs of the active variables, decisions as one word per variable (3 + the final ones)
    bool il; int n_groups; float* qc; unsigned* hardm[4];
    size_t bytes;
};

// The frame-interleaved family decodes batches that fill its groups of 32 frames (codes outside the exact families).
bool use_il(const qcldpc_code* code, int n_frames) {
    if (!code->il_ok || code->tune.il == 0) return false;
    if (code->tune.il == 2) return true;
    // (short columns too: the rate-1/10 stand-in, 10-11 edges per column, 0.340 against 0.367 ms per launch on 32 frames)
    const int groups = (n_frames + kIlGroup - 1) / kIlGroup;
    return n_frames >= 24 && 4 * n_frames >= 3 * groups * kIlGroup;      // at least 3/4 of the lanes carry a frame
}

Workspace carve(const qcldpc_code* code, int n_frames, void* base) {
    Workspace w;
    char* p = static_cast<char*>(base);
    size_t off = 0;
    w.il = use_il(code, n_frames);
    w.n_groups = (n_frames + kIlGroup - 1) / kIlGroup;
    w.qc = nullptr;
    for (int b = 0; b < 4; ++b) w.hardm[b] = nullptr;
    for (int b = 0; b < 3; ++b) w.hardbuf[b] = nullptr;
    const size_t fbytes = align_up((size_t)n_frames * sizeof(int), 256);
    if (w.il) {
        const size_t lines = (size_t)w.n_groups * kIlGroup * sizeof(float);            // bytes per line index
        const size_t qbytes = align_up(lines * code->n_act_edges * (code->Z + 1), 256);    // runs of Z lines + the halo line
        const size_t tbytes = align_up(lines * code->mb * (code->Z + 1), 256);
        const size_t cbytes = align_up(lines * code->n_act_cols * code->Z, 256);
        const size_t hbytes = align_up((size_t)w.n_groups * code->n_act_cols * code->Z * sizeof(unsigned), 256);
        for (int b = 0; b < 4; ++b) { w.qbuf[b] = reinterpret_cast<float*>(p + off); off += qbytes; }
        w.t = reinterpret_cast<float*>(p + off); off += tbytes;
        w.qc = reinterpret_cast<float*>(p + off); off += cbytes;
        for (int b = 0; b < 4; ++b) { w.hardm[b] = reinterpret_cast<unsigned*>(p + off); off += hbytes; }
    } else {
    const size_t qbytes = align_up((size_t)n_frames * code->n_act_edges * code->Zs * sizeof(float), 256);
    const size_t tbytes = align_up((size_t)n_frames * code->mb * code->Zs * sizeof(float), 256);
    const size_t hbytes = align_up((size_t)n_frames * code->n_act_cols * code->Zs, 256);
    for (int b = 0; b < 4; ++b) { w.qbuf[b] = reinterpret_cast<float*>(p + off); off += qbytes; }
    w.t = reinterpret_cast<float*>(p + off); off += tbytes;
    for (int b = 0; b < 3; ++b) { w.hardbuf[b] = reinterpret_cast<uint8_t*>(p + off); off += hbytes; }
    }
    w.done = reinterpret_cast<int*>(p + off); off += 2 * fbytes;       // two versions of n_frames ints, contiguous
    w.unsat = reinterpret_cast<int*>(p + off); off += fbytes;
    w.topbad = reinterpret_cast<int*>(p + off); off += 3 * fbytes;     // three slots of n_frames ints, contiguous
    w.fullbad = reinterpret_cast<int*>(p + off); off += fbytes;
    w.ticket = reinterpret_cast<unsigned*>(p + off); off += 256;
    w.bytes = off;
    return w;
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------------
// C ABI
// ---------------------------------------------------------------------------------------------------------------
extern "C" {

// The non-zero blocks of the base matrix: per base row the (column, shift) pairs, per base column the (row, shift)
// pairs, both in increasing index order.
struct BaseEntry { int idx, shift; };
struct BaseLists { std::vector<std::vector<BaseEntry>> rows, cols; };

static int code_from_lists(const BaseLists& B, int mb, int nb, int Z, qcldpc_code_t** out_code);

int qcldpc_code_create(const int32_t* base, int mb, int nb, int Z, qcldpc_code_t** out_code) {
    if (!base || !out_code || mb <= 0 || nb <= 0 || Z <= 0) return QCLDPC_ERR_BAD_ARGUMENT;
    *out_code = nullptr;
    BaseLists B;
    B.rows.resize(mb); B.cols.resize(nb);
    for (int R = 0; R < mb; ++R)
        for (int C = 0; C < nb; ++C) {
            const int p = base[(size_t)R * nb + C];
            if (p < -1 || p >= Z) return QCLDPC_ERR_BAD_ARGUMENT;
            if (p >= 0) { B.rows[R].push_back(BaseEntry{C, p}); B.cols[C].push_back(BaseEntry{R, p}); }
        }
    return code_from_lists(B, mb, nb, Z, out_code);
}

int qcldpc_code_create_sparse(const int32_t* rows, const int32_t* cols, const int32_t* shifts, int64_t n_entries,
                              int mb, int nb, int Z, qcldpc_code_t** out_code) {
    if (!out_code || mb <= 0 || nb <= 0 || Z <= 0 || n_entries < 0) return QCLDPC_ERR_BAD_ARGUMENT;
    if (n_entries > 0 && (!rows || !cols || !shifts)) return QCLDPC_ERR_BAD_ARGUMENT;
    *out_code = nullptr;
    BaseLists B;
    B.rows.resize(mb); B.cols.resize(nb);
    for (int64_t k = 0; k < n_entries; ++k) {
        if (rows[k] < 0 || rows[k] >= mb || cols[k] < 0 || cols[k] >= nb || shifts[k] < 0 || shifts[k] >= Z)
            return QCLDPC_ERR_BAD_ARGUMENT;
        B.rows[rows[k]].push_back(BaseEntry{cols[k], shifts[k]});
        B.cols[cols[k]].push_back(BaseEntry{rows[k], shifts[k]});
    }
    auto by_idx = [](const BaseEntry& a, const BaseEntry& b) { return a.idx < b.idx; };
    for (auto& r : B.rows) {
        std::sort(r.begin(), r.end(), by_idx);
        for (size_t k = 1; k < r.size(); ++k)
            if (r[k].idx == r[k - 1].idx) return QCLDPC_ERR_BAD_ARGUMENT;        // a block is ONE circulant
    }
    for (auto& c : B.cols) std::sort(c.begin(), c.end(), by_idx);
    return code_from_lists(B, mb, nb, Z, out_code);
}

static int code_from_lists(const BaseLists& B, int mb, int nb, int Z, qcldpc_code_t** out_code) {
    if ((int64_t)mb * Z > (int64_t)1 << 30 || (int64_t)nb * Z > (int64_t)1 << 30) return QCLDPC_ERR_UNSUPPORTED;
    qcldpc_code* code = new (std::nothrow) qcldpc_code();
    if (!code) return QCLDPC_ERR_ALLOC;
    code->mb = mb; code->nb = nb; code->Z = Z;
    code->n = (int64_t)nb * Z; code->m = (int64_t)mb * Z;

    // absorb at most one degree-1 column per row (the lowest-numbered one)
    std::vector<int> absorbed_by(nb, -1), n_active(mb, 0);
    code->row.assign(mb, RowDesc{0, 0, -1, 0, 0, 0, 0, 0});
    for (int R = 0; R < mb; ++R)
        for (const BaseEntry& e : B.rows[R])
            if (B.cols[e.idx].size() == 1 && code->row[R].abs_col < 0) {
                code->row[R].abs_col = e.idx;
                code->row[R].abs_shift = e.shift;
                absorbed_by[e.idx] = R;
            }
    for (int R = 0; R < mb; ++R)
        for (const BaseEntry& e : B.rows[R]) n_active[R] += absorbed_by[e.idx] < 0;
    code->filter_rows = false;
    for (int R = 0; R < mb; ++R) {
        const bool absorbed = code->row[R].abs_col >= 0;
        code->row[R].gen = (absorbed && n_active[R] == 2) ? 0 : (absorbed && n_active[R] == 3) ? 2 : 1;
        code->filter_rows = code->filter_rows || (code->row[R].abs_col < 0 && n_active[R] > 0);
    }

    // active columns and their edges: column by column, gen edges first (triple rows last among them), then pair
    // edges, each in row order
    struct HostEdge { int shift, row; };
    std::vector<HostEdge> edges;
    std::vector<int> act_index(nb, -1);
    std::vector<std::vector<int>> edge_of_row_entry(mb);        // parallel to B.rows[R]: active edge id or -1
    for (int R = 0; R < mb; ++R) edge_of_row_entry[R].assign(B.rows[R].size(), -1);
    auto row_pos = [&](int R, int C) {                           // position of column C in B.rows[R]
        const auto& r = B.rows[R];
        size_t lo = 0, hi = r.size();
        while (lo < hi) { const size_t mid = (lo + hi) / 2; if (r[mid].idx < C) lo = mid + 1; else hi = mid; }
        return lo;
    };
    code->max_dv = 0;
    for (int C = 0; C < nb; ++C) {
        if (absorbed_by[C] >= 0) continue;
        ColDesc cd{C, (int)edges.size(), 0, 0, 0, 0, 0, 0};
        for (int pass = 0; pass < 3; ++pass)
            for (const BaseEntry& e : B.cols[C]) {
                const int R = e.idx;
                if (code->row[R].gen != (pass == 0 ? 1 : pass == 1 ? 2 : 0)) continue;
                edge_of_row_entry[R][row_pos(R, C)] = (int)edges.size();
                edges.push_back(HostEdge{e.shift, R});
                ++cd.dv;
                cd.ng += pass < 2;
                cd.ngh += pass == 0;
            }
        act_index[C] = (int)code->col.size();
        code->col.push_back(cd);
        code->max_dv = std::max(code->max_dv, cd.dv);
    }
    code->n_act_cols = (int)code->col.size();
    code->n_act_edges = (int)edges.size();
    // kernel family: exact instantiations for the column shapes of the BASELINE.json codes (runs stored with a halo of
    // kHalo wrapped entries, common.cuh), else the generic kernel (compact runs, per-element wrap)
    bool uniform = code->n_act_cols > 0;
    for (const ColDesc& cd : code->col) uniform = uniform && cd.dv == code->col[0].dv && cd.ng == code->col[0].ng;
    const bool exact = uniform && code->n_act_cols <= kMaxExactCols && code->col[0].ng == 3 &&
                       (code->col[0].dv == 11 || code->col[0].dv == 21);
    code->halo = exact ? 1 : 0;
    code->Zs = exact ? (int)align_up((size_t)Z + kHalo, 32) : (int)align_up((size_t)Z, 8);   // whole 32-byte sectors
    const int Zs = code->Zs;
    // run offsets are formed as 32-bit BYTE offsets in the kernels: a frame's edge state and its static terms must each
    // stay below 2^30 floats
    if (code->max_dv > kMaxDv || (int64_t)code->n_act_edges * Zs >= ((int64_t)1 << 30) ||
        (int64_t)mb * Zs >= ((int64_t)1 << 30)) {
        delete code;
        return QCLDPC_ERR_UNSUPPORTED;
    }
    // row view
    for (int R = 0; R < mb; ++R) {
        code->row[R].ebeg = (int)code->redge.size();
        for (size_t k = 0; k < B.rows[R].size(); ++k) {
            const int e = edge_of_row_entry[R][k];
            const int C = B.rows[R][k].idx;
            if (e >= 0) code->redge.push_back(RowEdge{e, B.rows[R][k].shift, C, act_index[C]});
        }
        code->row[R].ne = (int)code->redge.size() - code->row[R].ebeg;
    }
    // per edge: where its partners are
    bool partners_ok = true;
    int max_np = 0;
    for (ColDesc& cd : code->col) {
        cd.gbeg = (int)code->gen.size();
        cd.pbeg = (int)code->partner.size();
        for (int k = 0; k < cd.dv; ++k) {
            const int e = cd.ebeg + k;
            const HostEdge& he = edges[e];
            const RowDesc& rd = code->row[he.row];
            EdgeDesc ed{he.shift, he.row * Zs, -1, 0, -1, 0};
            if (!rd.gen) {
                for (int j = 0; j < rd.ne; ++j) {
                    const RowEdge& re = code->redge[rd.ebeg + j];
                    if (re.edge == e) continue;
                    ed.p_off = re.edge * Zs;
                    ed.delta = ((re.shift - he.shift) % Z + Z) % Z;
                }
            } else {
                GenDesc gd{(int)code->partner.size() - cd.pbeg, rd.ne - 1, 0, 0};
                gd.counter = (rd.abs_col < 0 && code->redge[rd.ebeg].edge == e) ? 1 : 0;
                for (int j = 0; j < rd.ne; ++j) {
                    const RowEdge& re = code->redge[rd.ebeg + j];
                    if (re.edge == e) continue;
                    const PartnerDesc pd{re.edge * Zs, ((re.shift - he.shift) % Z + Z) % Z};
                    code->partner.push_back(pd);
                    if (rd.gen == 2) {                       // triple row: both partners also travel with the edge
                        if (ed.p_off < 0) { ed.p_off = pd.off; ed.delta = pd.delta; }
                        else { ed.p2_off = pd.off; ed.delta2 = pd.delta; }
                    }
                }
                code->gen.push_back(gd);
            }
            code->edge.push_back(ed);
        }
        cd.np = (int)code->partner.size() - cd.pbeg;
        max_np = std::max(max_np, cd.np);
        partners_ok = partners_ok && cd.np <= kMaxPartners;
    }
    if (!partners_ok) { delete code; return QCLDPC_ERR_UNSUPPORTED; }

    // kernel choice: exact instantiations for the column shapes of the BASELINE.json codes, else the generic one
    code->launcher = launch_pass_generic;
    code->max_np = max_np;
    if (exact) {
        code->launcher = code->col[0].dv == 11 ? launch_pass_dv11_ng3 : launch_pass_dv21_ng3;
        const ExactBuilder fill = code->col[0].dv == 11 ? launch_pass_dv11_ng3_table : launch_pass_dv21_ng3_table;
        const HostTables ht{code->edge.data(), code->gen.data(), code->partner.data(), code->col.data(),
                            code->n_act_cols};
        code->exact.resize(fill(ht, nullptr));
        fill(ht, code->exact.data());
    }
    code->tiles = (Z + kThreads - 1) / kThreads;
    {
        Tuning& tn = code->tune;
        const int v = env_int("QCLDPC_V", 0);
        tn.V = (v == 1 || v == 2) ? v : 0;
        tn.flip = env_int("QCLDPC_FLIP", 1) != 0;
        tn.merge_check = env_int("QCLDPC_MERGE_CHECK", 1) != 0;
        tn.cand_per_sm = std::max(0, env_int("QCLDPC_CAND_PER_SM", 0));
        tn.pack = env_int("QCLDPC_PACK", 1) != 0;
        const int fv = env_int("QCLDPC_FV", 0);
        tn.fv = (fv == 1 || fv == 2) ? fv : 0;
        const char* lp = getenv("QCLDPC_LOOP");
        tn.loop_graph = !(lp && strcmp(lp, "stream") == 0);
        tn.body_mult = std::min(16, std::max(0, env_int("QCLDPC_BODY", 0)));
        tn.il = std::min(2, std::max(0, env_int("QCLDPC_IL", 1)));
    }

    // frame-interleaved family: offsets in lines of 32 frames, runs of Z lines + one halo line (pass_il.cuh)
    const int Zp = Z + 1;
    code->edge_il = code->edge;
    for (EdgeDesc& d : code->edge_il) {
        d.t_off = d.t_off / Zs * Zp;
        if (d.p_off >= 0) d.p_off = d.p_off / Zs * Zp;
        if (d.p2_off >= 0) d.p2_off = d.p2_off / Zs * Zp;
    }
    code->partner_il = code->partner;
    for (PartnerDesc& d : code->partner_il) d.off = d.off / Zs * Zp;
    // byte offsets of lines within a group are signed 32-bit in the pass
    code->il_ok = !exact && code->n_act_cols > 0 && (int64_t)code->n_act_edges * Zp < ((int64_t)1 << 24) &&
                  (int64_t)mb * Zp < ((int64_t)1 << 24) &&
                  il_smem_bytes(code->max_dv, max_np, 2) <= (size_t)200 * 1024;
    // long columns (two warps per slot): the asynchronous variant -- messages in tensor memory, loads as asynchronous
    // copies through a ring, QCLDPC_ILA chunks deep (default 2; 0: register loads) --, eight variables per CTA so that
    // four CTAs share a multiprocessor; short columns: register loads
    code->il_w = il_pick_w(Z, code->max_dv, max_np);
    const bool long_cols = code->max_dv > 2 * kIlChunk;
    int as = long_cols ? env_int("QCLDPC_ILA", 2) : 0;
    if (as < 0 || as > 4) as = 0;
    if (as) code->il_w = std::min(8, 2 * ((Z + 1) / 2));
    if (const int wf = env_int("QCLDPC_ILW", 0)) {         // tuning knob: variables per CTA of k_pass_il (even, <= 12)
        if (wf >= 2 && wf <= (long_cols ? 12 : 24) && wf % 2 == 0 &&
            il_smem_bytes(code->max_dv, max_np, wf) <= (size_t)200 * 1024)
            code->il_w = wf;
    }
    // (the asynchronous variant: at most 10 warps per CTA -- 64 columns of tensor memory per warp, 256 per CTA)
    if (as && code->il_w <= 10 && il_smem_bytes(code->max_dv, max_np, code->il_w, as, code->il_w) <= (size_t)200 * 1024)
        code->il_as = as;
    else if (as)
        code->il_w = il_pick_w(Z, code->max_dv, max_np);
    if (code->il_ok) {                                     // one fixed-stride blob per column, in shared-memory layout
        const int mdv = std::max(code->max_dv, 1);
        const size_t stride = il_table_bytes(mdv, max_np);
        code->il_blob16 = (int)(stride / 16);
        code->il_blob.assign((size_t)code->n_act_cols * code->il_blob16, uint4{0, 0, 0, 0});
        for (int c = 0; c < code->n_act_cols; ++c) {
            const ColDesc& cd = code->col[c];
            char* base = reinterpret_cast<char*>(code->il_blob.data()) + (size_t)c * stride;
            IlColHdr hdr{cd.col, cd.ebeg, cd.dv, cd.ng, cd.ngh, cd.np, 0, 0};
            memcpy(base, &hdr, sizeof(hdr));
            IlEdgeA* ea = reinterpret_cast<IlEdgeA*>(base + sizeof(IlColHdr));
            GenDesc* eg = reinterpret_cast<GenDesc*>(ea + mdv);
            IlEdgeB* eb = reinterpret_cast<IlEdgeB*>(eg + mdv);
            IlRef* ep = reinterpret_cast<IlRef*>(eb + mdv);
            const IlRef none{0, 0};
            for (int k = 0; k < cd.dv; ++k) {
                const EdgeDesc& d = code->edge_il[cd.ebeg + k];
                // t_c of variable i is check (i - shift) mod Z; byte offsets of lines stay below 2^31 by il_ok
                ea[k] = IlEdgeA{il_ref(d.t_off, (Z - d.shift) % Z, Z), d.p_off >= 0 ? il_ref(d.p_off, d.delta, Z) : none};
                eb[k] = IlEdgeB{d.p2_off >= 0 ? il_ref(d.p2_off, d.delta2, Z) : none};
            }
            for (int k = 0; k < cd.ng; ++k) eg[k] = code->gen[cd.gbeg + k];
            for (int k = 0; k < cd.np; ++k) {
                const PartnerDesc& pd = code->partner_il[cd.pbeg + k];
                ep[k] = il_ref(pd.off, pd.delta, Z);
            }
        }
    }

    auto upload = [](auto& vec, auto** dptr) -> cudaError_t {
        const size_t bytes = std::max<size_t>(vec.size(), 1) * sizeof(vec[0]);
        cudaError_t e = cudaMalloc(reinterpret_cast<void**>(dptr), bytes);
        if (e != cudaSuccess) return e;
        if (!vec.empty()) e = cudaMemcpy(*dptr, vec.data(), vec.size() * sizeof(vec[0]), cudaMemcpyHostToDevice);
        return e;
    };
    cudaError_t e = upload(code->edge, &code->d_edge);
    if (e == cudaSuccess) e = upload(code->gen, &code->d_gen);
    if (e == cudaSuccess) e = upload(code->partner, &code->d_partner);
    if (e == cudaSuccess) e = upload(code->col, &code->d_col);
    if (e == cudaSuccess) e = upload(code->row, &code->d_row);
    if (e == cudaSuccess) e = upload(code->redge, &code->d_redge);
    if (e == cudaSuccess && code->il_ok) e = upload(code->edge_il, &code->d_edge_il);
    if (e == cudaSuccess && code->il_ok) e = upload(code->partner_il, &code->d_partner_il);
    if (e == cudaSuccess && code->il_ok) e = upload(code->il_blob, &code->d_il_blob);
    int dev = 0;
    if (e == cudaSuccess) e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&code->n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) { qcldpc_code_destroy(code); return cuda_fail(e, "qcldpc_code_create: table upload"); }
    *out_code = code;
    return QCLDPC_OK;
}

void qcldpc_code_destroy(qcldpc_code_t* code) {
    if (!code) return;
    for (GraphEntry& ge : code->graphs) cudaGraphExecDestroy(ge.exec);
    if (code->cap_main) cudaStreamDestroy(code->cap_main);
    if (code->cap_body) cudaStreamDestroy(code->cap_body);
    cudaFree(code->d_edge); cudaFree(code->d_gen); cudaFree(code->d_partner); cudaFree(code->d_col);
    cudaFree(code->d_row); cudaFree(code->d_redge);
    cudaFree(code->d_edge_il); cudaFree(code->d_partner_il); cudaFree(code->d_il_blob);
    delete code;
}

int qcldpc_code_info(const qcldpc_code_t* code, int64_t* n, int64_t* m, int64_t* active_base_edges) {
    if (!code) return QCLDPC_ERR_BAD_ARGUMENT;
    if (n) *n = code->n;
    if (m) *m = code->m;
    if (active_base_edges) *active_base_edges = code->n_act_edges;
    return QCLDPC_OK;
}

size_t qcldpc_workspace_bytes(const qcldpc_code_t* code, int n_frames) {
    if (!code || n_frames <= 0) return 0;
    return carve(code, n_frames, nullptr).bytes;
}

int qcldpc_decode(const qcldpc_code_t* code, const float* d_llr, const uint8_t* d_syndrome, int n_frames,
                  int max_iter, int early_stop, uint8_t* d_hard, int32_t* d_iters, uint8_t* d_pass,
                  float* d_posterior, void* d_workspace, size_t workspace_bytes, void* stream) {
    return qcldpc_decode_ex(code, d_llr, d_syndrome, n_frames, max_iter, early_stop, 1, d_hard, d_iters, d_pass,
                            d_posterior, d_workspace, workspace_bytes, stream);
}

// Two ways to run the iteration loop (same kernels, same results):
//   graph   (default) one CUDA graph per decode: prologue, the first few iterations, a conditional WHILE node whose
//           body is kLoopBody iterations + k_loop_ctl, epilogue.  The loop ends on the DEVICE when max_iter is reached or
//           when every frame has stopped, so a batch that has stopped issues at most one more body of (empty)
//           launches and the call still only enqueues.  Buffer rotation has period 12 (4 state buffers, 3 decision
//           buffers, 2 flag versions), so the body's kernel parameters are static; only the iteration NUMBER is read
//           from device memory (CheckArgs::t_base).  Instantiated graphs are cached in the handle by argument tuple.
//   stream  (QCLDPC_LOOP=stream, profiling on, or fewer iterations than one body) one launch per iteration from the
//           host; qcldpc_decode_host then polls the number of live frames every kPollEvery launches (host_poll).
namespace {

constexpr int kLoopBody = 12;
// A trip of the WHILE loop costs ~6 us on top of its launches (measured, B200): small batches, whose iterations take
// about that long, run bodies of 24 iterations, large ones bodies of 12 (a stopped batch then issues fewer empty launches).
inline int loop_body_len(const qcldpc_code* code, int n_frames) {
    const int mult = code->tune.body_mult ? code->tune.body_mult : (n_frames <= 8 ? 2 : 1);
    return kLoopBody * mult;
}

struct DecodePlan {
    const qcldpc_code* code;
    Workspace w;
    PassTables ptab; CheckTables ctab;
    InitArgs ia;
    PassLaunch pl;
    CheckArgs ca;
    int n_frames, max_iter, early_stop, check_from, cand_blocks, tiles1, fblocks;
    bool merge_check, flip;
    int* ctl;
    int32_t* d_iters; uint8_t* d_pass;
    bool il; IlLaunch ill;                               // frame-interleaved family (pass_il.cuh)

    int* done_ver(int t) const { return w.done + (size_t)(t & 1) * n_frames; }
    int* topbad_slot(int T) const { return w.topbad + (size_t)(((T % 3) + 3) % 3) * n_frames; }
    // the check is launched for iterations T >= check_from - 2: the filter slot of iteration I is dirty from pass I-2
    // and is cleared by the launch of iteration I-2, so the two launches before the first checked iteration only clear
    bool check_wanted(int T) const { return early_stop && T >= 1 && T >= check_from - 2; }
};

void issue_prologue(DecodePlan& P, cudaStream_t st) {
    k_reset<<<P.fblocks, 128, 0, st>>>(P.w.done, P.w.unsat, P.w.topbad, P.w.fullbad, P.w.ticket, P.d_iters, P.d_pass,
                                       P.n_frames, P.max_iter);
    ++g_launches;
    if (P.il) {
        launch_il_init(P.ill.tab, P.ctab, P.ill.args, st);
        g_launches += 2;
        return;
    }
    if (P.code->n_act_cols > 0) {
        k_init_cols<<<dim3(P.tiles1 * P.code->n_act_cols, P.n_frames), kThreads, 0, st>>>(P.ptab, P.ia);
        ++g_launches;
    }
    k_init_rows<<<dim3(P.tiles1 * P.code->mb, P.n_frames), kThreads, 0, st>>>(P.ctab, P.ia);
    ++g_launches;
}

// check of iteration T (+ *t_base), issued with launch t: reads the stopped-frame flags of version t & 1 (the ones pass
// t reads) and writes version (t + 1) & 1 for pass t+1
void set_check(DecodePlan& P, int T, int t, const int* t_base, const int* skip) {
    P.ca.t = T;
    P.ca.t_base = t_base;
    P.ca.skip = skip;
    P.ca.topbad = P.topbad_slot(T);
    P.ca.topbad_clear = P.topbad_slot(t);                // the slot pass t+1 writes (filter of iteration t)
    P.ca.done_r = P.done_ver(t);
    P.ca.done_w = P.done_ver(t + 1);
}

void launch_check(DecodePlan& P, cudaStream_t st, int T, int t, const int* t_base, const int* skip) {
    set_check(P, T, t, t_base, skip);
    const int pk = prof_begin(1, st);
    if (P.il) launch_il_cand(P.ctab, P.ca, P.ill.args, P.cand_blocks, st);
    else launch_pdl(k_cand, dim3(P.cand_blocks), dim3(kThreads), 0, st, P.ctab, P.ca);
    prof_end(pk, st);
    ++g_launches;
}

// Launch t = pass t carrying (or followed by) the early-exit check of iteration t-2 (check.cuh explains the lag).
// t_base != NULL: inside the WHILE body; t is then the launch's number in the FIRST trip of the loop, the real number is
// t + *t_base (the same modulo 12), and the check is always issued (the device decides whether it is due).
void issue_iteration(DecodePlan& P, cudaStream_t st, int t, const int* t_base) {
    const qcldpc_code* code = P.code;
    const bool want = t_base ? (P.early_stop != 0) : P.check_wanted(t - 2);
    const bool merged = P.merge_check && want && code->n_act_cols > 0;
    if (P.il) {
        IlLaunch& L = P.ill;
        L.stream = st;
        L.final_mode = false;
        L.args.q_in = P.w.qbuf[(t - 1) % 4]; L.args.q_out = P.w.qbuf[t % 4];
        L.args.hard_in = P.w.hardm[(t - 1) % 3]; L.args.hard_out = P.w.hardm[t % 3];
        L.args.topbad = P.topbad_slot(t - 1);
        L.args.done = P.done_ver(t);
        L.check = nullptr;
        if (merged) { set_check(P, t - 2, t, t_base, nullptr); L.check = &P.ca; }
        const int pk = prof_begin(0, st);
        launch_pass_il_entry(L);
        prof_end(pk, st);
        ++g_launches;
    } else if (code->n_act_cols > 0) {
        PassLaunch& pl = P.pl;
        pl.stream = st;
        pl.args.in_buf = (t - 1) % 4; pl.args.out_buf = t % 4;
        pl.args.flip = P.flip ? (t & 1) : 0;
        pl.args.hard_in = P.w.hardbuf[(t - 1) % 3]; pl.args.hard_out = P.w.hardbuf[t % 3];
        pl.args.topbad = P.topbad_slot(t - 1);
        pl.args.done = P.done_ver(t);
        pl.check_tab = nullptr; pl.check_args = nullptr;
        if (merged) {
            set_check(P, t - 2, t, t_base, nullptr);
            pl.check_tab = &P.ctab; pl.check_args = &P.ca;
        }
        const int pk = prof_begin(0, st);
        code->launcher(pl);
        prof_end(pk, st);
        ++g_launches;
    }
    if (want && !merged) launch_check(P, st, t - 2, t, t_base, nullptr);
}

// after the last launch t_last: the check of the last but one executed iteration (the last one is settled by
// k_check_final), then the outputs from each frame's frozen state: iteration d_iters[f] (= max_iter for the frames that
// did not stop)
void issue_epilogue(DecodePlan& P, cudaStream_t st, int t_last, const int* skip) {
    if (t_last >= 2 && P.check_wanted(t_last - 1)) launch_check(P, st, t_last - 1, t_last + 1, nullptr, skip);
    if (P.il) {
        IlLaunch& L = P.ill;
        L.stream = st;
        L.check = nullptr;
        L.args.hardm_final = P.w.hardm[0];               // max_iter = 0: the decisions of k_il_init_cols
        if (P.max_iter > 0) {
            L.args.hardm_final = P.w.hardm[3];
            L.final_mode = true;
            launch_pass_il_entry(L);
            L.final_mode = false;
            ++g_launches;
        }
        launch_il_check_final(P.ctab, L.args, st);
        k_flags_final<<<P.fblocks, 128, 0, st>>>(P.w.unsat, P.d_pass, P.n_frames);
        g_launches += 2;
        return;
    }
    if (P.code->n_act_cols > 0 && P.max_iter > 0) {
        P.pl.stream = st;
        P.pl.final_mode = true;
        P.pl.check_tab = nullptr; P.pl.check_args = nullptr;
        P.code->launcher(P.pl);
        P.pl.final_mode = false;
        ++g_launches;
    }
    set_check(P, 0, 0, nullptr, nullptr);
    k_check_final<<<dim3(P.tiles1 * P.code->mb, P.n_frames), kThreads, 0, st>>>(P.ctab, P.ca);
    k_flags_final<<<P.fblocks, 128, 0, st>>>(P.w.unsat, P.d_pass, P.n_frames);
    g_launches += 2;
}

// Captures the whole decode into a graph with a conditional WHILE node around the bulk of the iterations.
// Returns cudaSuccess and the instantiated graph, or the error (the caller then runs the stream path).
cudaError_t build_decode_graph(DecodePlan& P, cudaGraphExec_t* exec_out) {
    qcldpc_code* code = const_cast<qcldpc_code*>(P.code);          // the capture streams live in the handle (under graph_mu)
    cudaError_t e = cudaSuccess;
    if (!code->cap_main) e = cudaStreamCreateWithFlags(&code->cap_main, cudaStreamNonBlocking);
    if (e == cudaSuccess && !code->cap_body) e = cudaStreamCreateWithFlags(&code->cap_body, cudaStreamNonBlocking);
    if (e != cudaSuccess) return e;
    if (P.il) {                                                   // kernel attributes are set outside the capture
        P.ill.prepare_only = 1;
        launch_pass_il_entry(P.ill);
        P.ill.prepare_only = 0;
    } else if (code->n_act_cols > 0) {
        P.pl.prepare_only = 1;
        P.pl.final_mode = false; code->launcher(P.pl);
        P.pl.final_mode = true; code->launcher(P.pl);
        P.pl.final_mode = false;
        P.pl.prepare_only = 0;
    }
    const int body = loop_body_len(code, P.n_frames);
    int pre = P.max_iter % body;
    if (pre < 2) pre += body;                                     // every launch of the body carries a check of T >= 1
    const int loops = (P.max_iter - pre) / body;                  // > 0: the caller made sure
    int* const iter_base = P.ctl + kCtlIterBase;
    const int* const stopped = P.ctl + kCtlStopped;

    cudaStream_t cm = code->cap_main, cb = code->cap_body;
    e = cudaStreamBeginCapture(cm, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) return e;
    cudaGraph_t graph = nullptr;
    bool body_open = false;
    auto bail = [&](cudaError_t err) {
        cudaGraph_t g = nullptr;
        if (body_open) cudaStreamEndCapture(cb, &g);
        g = nullptr;
        cudaStreamEndCapture(cm, &g);
        if (g) cudaGraphDestroy(g);
        cudaGetLastError();
        return err;
    };
    issue_prologue(P, cm);
    for (int t = 1; t <= pre; ++t) issue_iteration(P, cm, t, nullptr);
    {
        cudaStreamCaptureStatus status;
        const cudaGraphNode_t* deps = nullptr;
        size_t n_deps = 0;
        e = cudaStreamGetCaptureInfo(cm, &status, nullptr, &graph, &deps, &n_deps);
        if (e != cudaSuccess || status != cudaStreamCaptureStatusActive) return bail(e != cudaSuccess ? e : cudaErrorUnknown);
        cudaGraphConditionalHandle handle;
        e = cudaGraphConditionalHandleCreate(&handle, graph, 1, cudaGraphCondAssignDefault);
        if (e != cudaSuccess) return bail(e);
        cudaGraphNodeParams np = {};
        np.type = cudaGraphNodeTypeConditional;
        np.conditional.handle = handle;
        np.conditional.type = cudaGraphCondTypeWhile;
        np.conditional.size = 1;
        cudaGraphNode_t loop_node;
        e = cudaGraphAddNode(&loop_node, graph, deps, n_deps, &np);
        if (e != cudaSuccess) return bail(e);
        cudaGraph_t body_graph = np.conditional.phGraph_out[0];
        e = cudaStreamUpdateCaptureDependencies(cm, &loop_node, 1, cudaStreamSetCaptureDependencies);
        if (e != cudaSuccess) return bail(e);
        e = cudaStreamBeginCaptureToGraph(cb, body_graph, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal);
        if (e != cudaSuccess) return bail(e);
        body_open = true;
        for (int j = 1; j <= body; ++j) issue_iteration(P, cb, pre + j, iter_base);
        k_loop_ctl<<<1, 1, 0, cb>>>(handle, P.ctl, body, loops * body, pre);
        ++g_launches;
        cudaGraph_t g2 = nullptr;
        e = cudaStreamEndCapture(cb, &g2);
        body_open = false;
        if (e != cudaSuccess) return bail(e);
    }
    issue_epilogue(P, cm, P.max_iter, stopped);
    e = cudaStreamEndCapture(cm, &graph);
    if (e != cudaSuccess) { cudaGetLastError(); return e; }
    e = cudaGraphInstantiate(exec_out, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) cudaGetLastError();
    return e;
}

bool same_key(const GraphKey& a, const GraphKey& b) {
    return a.llr == b.llr && a.syn == b.syn && a.hard == b.hard && a.iters == b.iters && a.pass == b.pass &&
           a.post == b.post && a.ws == b.ws && a.n_frames == b.n_frames && a.max_iter == b.max_iter &&
           a.early_stop == b.early_stop && a.check_from == b.check_from && a.device == b.device;
}

}  // namespace

static int decode_impl(const qcldpc_code_t* code, const float* d_llr, const uint8_t* d_syndrome, int n_frames,
                       int max_iter, int early_stop, int check_from_iter, uint8_t* d_hard, int32_t* d_iters,
                       uint8_t* d_pass, float* d_posterior, void* d_workspace, size_t workspace_bytes, void* stream,
                       bool host_poll, bool allow_graph = true);

int qcldpc_decode_ex(const qcldpc_code_t* code, const float* d_llr, const uint8_t* d_syndrome, int n_frames,
                     int max_iter, int early_stop, int check_from_iter, uint8_t* d_hard, int32_t* d_iters,
                     uint8_t* d_pass, float* d_posterior, void* d_workspace, size_t workspace_bytes, void* stream) {
    return decode_impl(code, d_llr, d_syndrome, n_frames, max_iter, early_stop, check_from_iter, d_hard, d_iters,
                       d_pass, d_posterior, d_workspace, workspace_bytes, stream, false);
}

static int decode_impl(const qcldpc_code_t* code, const float* d_llr, const uint8_t* d_syndrome, int n_frames,
                       int max_iter, int early_stop, int check_from_iter, uint8_t* d_hard, int32_t* d_iters,
                       uint8_t* d_pass, float* d_posterior, void* d_workspace, size_t workspace_bytes, void* stream,
                       bool host_poll, bool allow_graph) {
    constexpr int kPollEvery = 32;
    g_launches = 0;
    if (check_from_iter < 1) return QCLDPC_ERR_BAD_ARGUMENT;
    if (!code || !d_llr || !d_syndrome || !d_hard || !d_iters || !d_pass) return QCLDPC_ERR_BAD_ARGUMENT;
    if (n_frames <= 0 || n_frames > QCLDPC_MAX_FRAMES || max_iter < 0) return QCLDPC_ERR_BAD_ARGUMENT;
    if (!d_workspace || (reinterpret_cast<uintptr_t>(d_workspace) & 255) ||
        workspace_bytes < qcldpc_workspace_bytes(code, n_frames))
        return QCLDPC_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    DecodePlan P;
    P.code = code;
    P.w = carve(code, n_frames, d_workspace);
    const Workspace& w = P.w;
    const int Z = code->Z, Zs = code->Zs;
    const int64_t EZs = (int64_t)code->n_act_edges * Zs, mZs = (int64_t)code->mb * Zs;
    const int64_t AZs = (int64_t)code->n_act_cols * Zs;
    P.tiles1 = (Z + kThreads - 1) / kThreads;
    P.fblocks = (n_frames + 127) / 128;
    P.ptab = PassTables{code->d_edge, code->d_gen, code->d_partner, code->d_col};
    P.ctab = CheckTables{code->d_row, code->d_redge};
    P.n_frames = n_frames; P.max_iter = max_iter; P.early_stop = early_stop; P.check_from = check_from_iter;
    P.d_iters = d_iters; P.d_pass = d_pass;
    P.ctl = reinterpret_cast<int*>(w.ticket);
    P.ia = InitArgs{d_llr, d_syndrome, w.qbuf[0], w.t, w.hardbuf[0], d_hard, d_posterior,
                    Z, Zs, P.tiles1, code->halo, code->n, code->m, EZs, mZs, AZs};

    // exact families: two variables per thread (1 KB windows) once the grid still fills the chip several times over;
    // small batches keep one variable per thread (more CTAs in flight).  Tuning::V overrides.
    int V = 1;
    if (!code->exact.empty()) {
        const int64_t ctas_v2 = (int64_t)((Z + 2 * kThreads - 1) / (2 * kThreads)) * code->n_act_cols * n_frames;
        if (ctas_v2 >= (int64_t)4 * 8 * code->n_sm) V = 2;
        if (code->tune.V) V = code->tune.V;
    }
    P.flip = code->tune.flip != 0;
    const int fv = code->tune.fv ? code->tune.fv : (n_frames >= 4 ? 2 : 1);   // generic pass: frames per thread
    P.pl = PassLaunch{P.ptab,
                      PassArgs{d_llr, {w.qbuf[0], w.qbuf[1], w.qbuf[2], w.qbuf[3]}, w.t, nullptr, nullptr, d_hard, d_posterior,
                               w.done, d_iters, nullptr, 0, 0, Z, Zs, code->tiles, 0, 0, n_frames, -1, code->n, EZs, mZs, AZs},
                      st, V, false,
                      code->exact.empty() ? nullptr : code->exact.data(), nullptr, nullptr, code->n_act_cols, n_frames,
                      code->max_np, code->max_dv, code->n_sm, fv, code->tune.pack, 0};
    P.ca = CheckArgs{d_llr, d_syndrome, {w.qbuf[0], w.qbuf[1], w.qbuf[2], w.qbuf[3]},
                     {w.hardbuf[0], w.hardbuf[1], w.hardbuf[2]}, d_hard,
                     d_posterior, w.done, w.done, d_iters, d_pass, nullptr, nullptr, w.fullbad, w.unsat, w.ticket,
                     n_frames, code->mb, Z, Zs, P.tiles1, 0, check_from_iter, code->n, code->m, EZs, AZs,
                     nullptr, P.ctl + kCtlNLive, nullptr};
    // early-exit grid: persistent; small batches are launch-bound and almost never have a candidate, so a smaller grid
    // (less to schedule and retire between two passes) wins there
    const int cand_per_sm = code->tune.cand_per_sm ? code->tune.cand_per_sm : (n_frames <= 8 ? 1 : 4);
    P.cand_blocks = std::max(1, std::min(code->n_sm * cand_per_sm, code->mb * P.tiles1));
    P.merge_check = code->tune.merge_check != 0;
    P.il = w.il;
    if (P.il) {
        const int64_t EZ = (int64_t)code->n_act_edges * (Z + 1), mZ = (int64_t)code->mb * (Z + 1),
                      AZ = (int64_t)code->n_act_cols * Z;
        IlArgs ia{};
        ia.llr = d_llr; ia.syn = d_syndrome;
        for (int b = 0; b < 4; ++b) ia.qb[b] = w.qbuf[b];
        ia.t = w.t; ia.qc = w.qc;
        for (int b = 0; b < 3; ++b) ia.hardm[b] = w.hardm[b];
        ia.hardm_final = w.hardm[3];
        ia.d_hard = d_hard; ia.d_post = d_posterior;
        ia.done = w.done; ia.iters = d_iters; ia.topbad = nullptr; ia.unsat = w.unsat;
        ia.Z = Z; ia.Zp = Z + 1; ia.W = code->il_w;
        ia.spc = (Z + 1) / 2; ia.ipc = std::min(code->il_w / 2, ia.spc);
        ia.as_depth = code->il_as;
        ia.n_frames = n_frames; ia.n_groups = w.n_groups; ia.n_cols = code->n_act_cols; ia.mb = code->mb;
        ia.cand_x = -1; ia.split = code->max_dv > 16 ? 4 : 1; ia.max_dv = std::max(code->max_dv, 1);
        ia.max_np = code->max_np;
        ia.blob = code->d_il_blob; ia.blob16 = code->il_blob16;
        ia.n = code->n; ia.m = code->m; ia.EZ = EZ; ia.mZ = mZ; ia.AZ = AZ;
        P.ill = IlLaunch{PassTables{code->d_edge_il, code->d_gen, code->d_partner_il, code->d_col}, P.ctab, ia, st,
                         nullptr, false, code->n_sm, 0};
        P.cand_blocks = std::max(1, std::min(code->n_sm * 2, code->mb * Z / 8 + 1));
    }

    // ---- graph path
    const int body = loop_body_len(code, n_frames);
    // (a caller that is itself capturing `stream` into a graph gets the plain launches: they become nodes of ITS graph)
    cudaStreamCaptureStatus caller_capture = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &caller_capture) != cudaSuccess) { cudaGetLastError(); caller_capture = cudaStreamCaptureStatusNone; }
    if (allow_graph && code->tune.loop_graph && g_prof.stride == 0 && max_iter >= body + 2 &&
        caller_capture == cudaStreamCaptureStatusNone) {
        int dev = 0;
        CUDA_TRY(cudaGetDevice(&dev));
        const GraphKey key{d_llr, d_syndrome, d_hard, d_iters, d_pass, d_posterior, d_workspace,
                           n_frames, max_iter, early_stop, check_from_iter, dev};
        qcldpc_code* mc = const_cast<qcldpc_code*>(code);
        std::lock_guard<std::mutex> lock(mc->graph_mu);
        cudaGraphExec_t exec = nullptr;
        for (GraphEntry& ge : mc->graphs)
            if (same_key(ge.key, key)) { exec = ge.exec; ge.stamp = ++mc->graph_clock; break; }
        if (!exec) {
            const cudaError_t e = build_decode_graph(P, &exec);
            if (e != cudaSuccess) {
                exec = nullptr;
                snprintf(g_cuda_error, sizeof(g_cuda_error), "graph loop unavailable (%s): stream loop used",
                         cudaGetErrorString(e));
                g_launches = 0;
            } else {
                if (mc->graphs.size() >= 8) {                    // evict the least recently used entry
                    size_t old = 0;
                    for (size_t k = 1; k < mc->graphs.size(); ++k)
                        if (mc->graphs[k].stamp < mc->graphs[old].stamp) old = k;
                    cudaGraphExecDestroy(mc->graphs[old].exec);  // a launch in flight completes first
                    mc->graphs.erase(mc->graphs.begin() + old);
                }
                mc->graphs.push_back(GraphEntry{key, exec, ++mc->graph_clock});
            }
        }
        if (exec) {
            CUDA_TRY(cudaGraphLaunch(exec, st));
            g_loop_mode = 1;
            return QCLDPC_OK;
        }
    }

    // ---- stream path
    g_loop_mode = 0;
    issue_prologue(P, st);
    int t_last = 0;                                      // last launch issued
    for (int t = 1; t <= max_iter; ++t) {
        issue_iteration(P, st, t, nullptr);
        t_last = t;
        if (host_poll && early_stop && t % kPollEvery == 0 && t < max_iter) {
            int* const d_live = P.ctl + kCtlLive;
            int live = 1;
            k_live_count<<<1, 128, 0, st>>>(P.check_wanted(t - 2) ? P.done_ver(t + 1) : P.done_ver(t), n_frames, d_live);
            ++g_launches;
            CUDA_TRY(cudaMemcpyAsync(&live, d_live, sizeof(int), cudaMemcpyDeviceToHost, st));
            CUDA_TRY(cudaStreamSynchronize(st));
            if (live == 0) break;                        // every frame is frozen: the remaining launches would be empty
        }
    }
    k_set_int<<<1, 1, 0, st>>>(P.ctl + kCtlIssued, t_last);
    ++g_launches;
    issue_epilogue(P, st, t_last, nullptr);
    CUDA_TRY(cudaGetLastError());
    return QCLDPC_OK;
}

int qcldpc_iterations_issued(const qcldpc_code_t* code, int n_frames, const void* d_workspace, void* stream,
                             int* h_iterations) {
    if (!code || n_frames <= 0 || !d_workspace || !h_iterations) return QCLDPC_ERR_BAD_ARGUMENT;
    const Workspace w = carve(code, n_frames, const_cast<void*>(d_workspace));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    CUDA_TRY(cudaMemcpyAsync(h_iterations, reinterpret_cast<const int*>(w.ticket) + kCtlIssued, sizeof(int),
                             cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return QCLDPC_OK;
}

int qcldpc_last_loop_mode(void) { return g_loop_mode; }

// ---- decode without any allocation: the workspace is a file-scope device array ------------------------------------
// (every GPU that loads the library holds QCLDPC_STATIC_WORKSPACE_BYTES of it until the process exits)
static __device__ __align__(256) unsigned char g_static_workspace[QCLDPC_STATIC_WORKSPACE_BYTES];

namespace {
// In host code `g_static_workspace` is a host-side stand-in, not a device address: the address a kernel may use comes
// from cudaGetSymbolAddress, asked once per device with that device current.
constexpr int kMaxStaticDevices = 64;
void* g_static_ws_ptr[kMaxStaticDevices] = {};
std::mutex g_static_ws_mu;

int static_workspace_ptr(void** out) {
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxStaticDevices) {
        snprintf(g_cuda_error, sizeof(g_cuda_error), "qcldpc_decode_static: device ordinal %d beyond %d", dev,
                 kMaxStaticDevices - 1);
        return QCLDPC_ERR_UNSUPPORTED;
    }
    std::lock_guard<std::mutex> lock(g_static_ws_mu);
    if (!g_static_ws_ptr[dev]) {
        void* ptr = nullptr;
        CUDA_TRY(cudaGetSymbolAddress(&ptr, g_static_workspace));
        if (!ptr || (reinterpret_cast<uintptr_t>(ptr) & 255)) {
            snprintf(g_cuda_error, sizeof(g_cuda_error), "qcldpc_decode_static: bad address of the static workspace");
            return QCLDPC_ERR_CUDA;
        }
        g_static_ws_ptr[dev] = ptr;
    }
    *out = g_static_ws_ptr[dev];
    return QCLDPC_OK;
}
}  // namespace

size_t qcldpc_static_workspace_bytes(void) { return (size_t)QCLDPC_STATIC_WORKSPACE_BYTES; }

int qcldpc_decode_static(const qcldpc_code_t* code, const float* d_llr, const uint8_t* d_syndrome, int n_frames,
                         int max_iter, int early_stop, int check_from_iter, uint8_t* d_hard, int32_t* d_iters,
                         uint8_t* d_pass, float* d_posterior, void* stream) {
    if (!code || n_frames <= 0 || n_frames > QCLDPC_MAX_FRAMES) return QCLDPC_ERR_BAD_ARGUMENT;
    const size_t need = qcldpc_workspace_bytes(code, n_frames);
    if (need == 0 || need > (size_t)QCLDPC_STATIC_WORKSPACE_BYTES) {
        snprintf(g_cuda_error, sizeof(g_cuda_error),
                 "qcldpc_decode_static: this code and batch need %zu bytes of workspace, the static workspace holds %zu: "
                 "use qcldpc_decode with a workspace of the caller's", need, (size_t)QCLDPC_STATIC_WORKSPACE_BYTES);
        return QCLDPC_ERR_WORKSPACE;
    }
    if (g_prof.stride != 0) {                                 // the profile's event pool grows by cudaEventCreate
        snprintf(g_cuda_error, sizeof(g_cuda_error), "qcldpc_decode_static: not while qcldpc_profile_enable is on");
        return QCLDPC_ERR_BAD_ARGUMENT;
    }
    void* ws = nullptr;
    const int rc = static_workspace_ptr(&ws);
    if (rc != QCLDPC_OK) return rc;
    // plain launches, one pass per iteration, no graph (building one allocates), no host polling; the prologue
    // (k_reset and the init kernels) clears and rewrites everything of the workspace that a decode reads
    return decode_impl(code, d_llr, d_syndrome, n_frames, max_iter, early_stop, check_from_iter, d_hard, d_iters, d_pass,
                       d_posterior, ws, (size_t)QCLDPC_STATIC_WORKSPACE_BYTES, stream, false, false);
}

size_t qcldpc_host_workspace_bytes(const qcldpc_code_t* code, int n_frames, int want_posterior) {
    if (!code || n_frames <= 0) return 0;
    size_t b = qcldpc_workspace_bytes(code, n_frames);
    b += align_up((size_t)n_frames * code->n * sizeof(float), 256);      // llr
    b += align_up((size_t)n_frames * code->m, 256);                      // syndrome
    b += align_up((size_t)n_frames * code->n, 256);                      // hard
    b += align_up((size_t)n_frames * sizeof(int32_t), 256);              // iters
    b += align_up((size_t)n_frames, 256);                                // pass
    if (want_posterior) b += align_up((size_t)n_frames * code->n * sizeof(float), 256);
    return b;
}

int qcldpc_decode_host(const qcldpc_code_t* code, const float* h_llr, const uint8_t* h_syndrome, int n_frames,
                       int max_iter, int early_stop, uint8_t* h_hard, int32_t* h_iters, uint8_t* h_pass,
                       float* h_posterior, void* d_workspace, size_t workspace_bytes, void* stream) {
    return qcldpc_decode_host_ex(code, h_llr, h_syndrome, n_frames, max_iter, early_stop, 1, h_hard, h_iters, h_pass,
                                 h_posterior, d_workspace, workspace_bytes, stream);
}

int qcldpc_decode_host_ex(const qcldpc_code_t* code, const float* h_llr, const uint8_t* h_syndrome, int n_frames,
                          int max_iter, int early_stop, int check_from_iter, uint8_t* h_hard, int32_t* h_iters,
                          uint8_t* h_pass, float* h_posterior, void* d_workspace, size_t workspace_bytes,
                          void* stream) {
    g_launches = 0;
    if (!code || !h_llr || !h_syndrome || !h_hard || !h_iters || !h_pass) return QCLDPC_ERR_BAD_ARGUMENT;
    if (n_frames <= 0 || n_frames > QCLDPC_MAX_FRAMES || max_iter < 0 || check_from_iter < 1)
        return QCLDPC_ERR_BAD_ARGUMENT;
    if (!d_workspace || (reinterpret_cast<uintptr_t>(d_workspace) & 255) ||
        workspace_bytes < qcldpc_host_workspace_bytes(code, n_frames, h_posterior != nullptr))
        return QCLDPC_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    char* p = static_cast<char*>(d_workspace);
    const size_t core = qcldpc_workspace_bytes(code, n_frames);
    size_t off = core;
    const size_t llr_b = (size_t)n_frames * code->n * sizeof(float), syn_b = (size_t)n_frames * code->m;
    const size_t hard_b = (size_t)n_frames * code->n;
    float* d_llr = reinterpret_cast<float*>(p + off); off += align_up(llr_b, 256);
    uint8_t* d_syn = reinterpret_cast<uint8_t*>(p + off); off += align_up(syn_b, 256);
    uint8_t* d_hard = reinterpret_cast<uint8_t*>(p + off); off += align_up(hard_b, 256);
    int32_t* d_iters = reinterpret_cast<int32_t*>(p + off); off += align_up((size_t)n_frames * sizeof(int32_t), 256);
    uint8_t* d_pass = reinterpret_cast<uint8_t*>(p + off); off += align_up((size_t)n_frames, 256);
    float* d_post = nullptr;
    if (h_posterior) { d_post = reinterpret_cast<float*>(p + off); off += align_up(llr_b, 256); }
    CUDA_TRY(cudaMemcpyAsync(d_llr, h_llr, llr_b, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(d_syn, h_syndrome, syn_b, cudaMemcpyHostToDevice, st));
    const int rc = decode_impl(code, d_llr, d_syn, n_frames, max_iter, early_stop, check_from_iter, d_hard, d_iters,
                               d_pass, d_post, d_workspace, core, stream, true);
    if (rc != QCLDPC_OK) return rc;
    CUDA_TRY(cudaMemcpyAsync(h_hard, d_hard, hard_b, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(h_iters, d_iters, (size_t)n_frames * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(h_pass, d_pass, (size_t)n_frames, cudaMemcpyDeviceToHost, st));
    if (h_posterior) CUDA_TRY(cudaMemcpyAsync(h_posterior, d_post, llr_b, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return QCLDPC_OK;
}

int64_t qcldpc_last_launch_count(void) { return g_launches; }

int qcldpc_profile_enable(int stride) {
    if (stride < 0) return QCLDPC_ERR_BAD_ARGUMENT;
    g_prof.stride = stride;
    g_prof.kind.clear();
    g_prof.launched[0] = g_prof.launched[1] = 0;
    if (stride == 0) {                                     // switching it off releases the event pool
        for (cudaEvent_t ev : g_prof.pool) cudaEventDestroy(ev);
        g_prof.pool.clear();
        g_prof.pool.shrink_to_fit();
    }
    return QCLDPC_OK;
}

int qcldpc_profile_collect(double* ms_sum, int64_t* timed, int64_t* launched) {
    if (!ms_sum || !timed || !launched) return QCLDPC_ERR_BAD_ARGUMENT;
    Profile& p = g_prof;
    for (int k = 0; k < 2; ++k) { ms_sum[k] = 0.0; timed[k] = 0; launched[k] = p.launched[k]; }
    for (size_t k = 0; k < p.kind.size(); ++k) {
        CUDA_TRY(cudaEventSynchronize(p.pool[2 * k + 1]));
        float ms = 0.0f;
        CUDA_TRY(cudaEventElapsedTime(&ms, p.pool[2 * k], p.pool[2 * k + 1]));
        ms_sum[p.kind[k]] += ms;
        timed[p.kind[k]] += 1;
    }
    p.kind.clear();
    p.launched[0] = p.launched[1] = 0;
    return QCLDPC_OK;
}

const char* qcldpc_status_string(int status) {
    switch (status) {
        case QCLDPC_OK: return "ok";
        case QCLDPC_ERR_BAD_ARGUMENT: return "bad argument";
        case QCLDPC_ERR_UNSUPPORTED:
            return "unsupported code (active column degree > 64, gen-row partner table or size out of range)";
        case QCLDPC_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
        case QCLDPC_ERR_CUDA: return "CUDA runtime error";
        case QCLDPC_ERR_ALLOC: return "host allocation failed";
        default: return "unknown status";
    }
}

const char* qcldpc_last_cuda_error(void) { return g_cuda_error; }

}  // extern "C"

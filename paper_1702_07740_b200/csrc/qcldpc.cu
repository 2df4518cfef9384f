// libqcldpc -- B200 (sm_100a) flooding Sum-Product decoder for QC-LDPC codes in syndrome form.
// C ABI: include/qcldpc.h.  Design notes: DESIGN.md.  Citations "P:NNN" are /root/reference/PAPER.md lines.
//
// Arithmetic domain.  Edge state is stored as  q_vc = sgn(L_vc) * exp(-|L_vc|)  (sign in the IEEE sign bit).
// With tanh(|L|/2) = (1-q)/(1+q) the paper's check-node rule
//     |m_cv| = Phi^-1( sum_{v'} Phi(|L_v'c|) ) = 2 atanh( prod_{v'} tanh(|L_v'c|/2) )
// becomes a Moebius ("velocity") addition of the q's,  q_a [+] q_b = (q_a + q_b) / (1 + q_a q_b),
// and |m_cv| = -ln( [+]_{v' in N(c)\v} q_v'c ).  Keeping numerator and denominator apart,
//     (num, den) <- (num + a*den, den + a*num),   |m_cv| = ln den - ln num,
// needs no division, no cancellation (all terms are >= 0) and one ex2 + two lg2 per edge and iteration.
// Degree-1 variables that are absorbed into their row contribute a constant q, folded together with the
// syndrome sign (-1)^{s_c} (reading S1) into one static float per check, t_c.
//
// Kernels (one thread per unit, frames on blockIdx.y so that the sweep is frame-major and a frame's working set
// stays in the 126 MB L2 while it is being processed):
//   k_init_q   a0  q^(0) = q(Q_v) on every active edge; hard/posterior of active variables at t = 0
//   k_init_t   a0  t_c from the absorbed variable's LLR and the syndrome bit
//   k_vn_pass  a1+a2  fused check-node + variable-node update, VN-centric: the thread of active variable v gathers,
//              for each of its edges (c,v), the q of the OTHER edges of c (+ t_c), forms m_cv, then L_v, xhat_v and
//              all L_vc by prefix/suffix sums (direct exclusion, no total-minus-self), and writes q^(t) (ping-pong)
//   k_check    a3  check-centric: decides the absorbed degree-1 variables (L_j = Q_j + m_cj), xhat parity vs s_c,
//              per-frame count of unsatisfied checks (integer atomics only); optional posterior write
//   k_flags    a3  per-frame early exit: freezes d_iters / d_pass / done
#include "common.cuh"

#include <algorithm>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

namespace qc {
// one object file per instantiation of k_vn_pass (vn_inst.cu)
void launch_vn_dv8(const VnLaunch&);
void launch_vn_dv11(const VnLaunch&);
void launch_vn_dv16(const VnLaunch&);
void launch_vn_dv21(const VnLaunch&);
void launch_vn_dv32(const VnLaunch&);
void launch_vn_dv64(const VnLaunch&);
}  // namespace qc

using namespace qc;

namespace {

thread_local char g_cuda_error[512] = "";
thread_local int64_t g_launches = 0;

// Optional launch timing (qcldpc_profile_enable): CUDA event pairs around sampled launches, on the decode stream.
struct Profile {
    int stride = 0;                       // 0 = off
    std::vector<cudaEvent_t> pool;        // reused across calls
    std::vector<int> kind;                // kind of pair k (events 2k, 2k+1)
    int64_t launched[2] = {0, 0};
};
thread_local Profile g_prof;

}  // namespace

struct qcldpc_code {
    int mb, nb, Z;
    int64_t n, m;
    int n_act_cols, n_act_edges, n_partners, max_dv, bucket;
    bool uniform_dv, inline_ok;
    std::vector<PairDesc> pair;
    std::vector<PartnerDesc> partner;
    std::vector<GenDesc> gen;
    std::vector<ColDesc> col;
    std::vector<RowDesc> row;
    std::vector<RowEdge> redge;
    // device copies
    PairDesc* d_pair = nullptr; PartnerDesc* d_partner = nullptr; GenDesc* d_gen = nullptr; ColDesc* d_col = nullptr;
    RowDesc* d_row = nullptr; RowEdge* d_redge = nullptr;
    VnTablesInline vn_inl; CnTablesInline cn_inl;
    VnLauncher launcher = nullptr;
};

namespace {

struct InitArgs {
    const float* llr; const uint8_t* syn; float* q0; float* t; uint8_t* hard; float* post;
    int Z, tiles; int64_t n, m, EZ;
};

// a0: q^(0) on every active edge, decisions at t = 0 for active variables
template <class Tables>
__global__ void __launch_bounds__(kThreads) k_init_q(const __grid_constant__ Tables tab, const InitArgs a) {
    const int f = blockIdx.y;
    const int ca = blockIdx.x / a.tiles;
    const int i = (blockIdx.x - ca * a.tiles) * kThreads + threadIdx.x;
    if (i >= a.Z) return;
    const ColDesc cd = tab.col[ca];
    const int64_t v = (int64_t)cd.col * a.Z + i;
    const float Q = __ldg(a.llr + (int64_t)f * a.n + v);
    const float q = q_of_llr(Q);
    float* q0 = a.q0 + (int64_t)f * a.EZ;
    for (int k = 0; k < cd.dv; ++k) q0[(int64_t)(cd.ebeg + k) * a.Z + i] = q;
    a.hard[(int64_t)f * a.n + v] = Q < 0.0f ? 1 : 0;
    if (a.post) a.post[(int64_t)f * a.n + v] = Q;
}

// a0: t_c = (-1)^{s_c} sgn(Q_j) exp(-|Q_j|) for the absorbed variable j of check c, or (-1)^{s_c} * 0
template <class Tables>
__global__ void __launch_bounds__(kThreads) k_init_t(const __grid_constant__ Tables tab, const InitArgs a) {
    const int f = blockIdx.y;
    const int R = blockIdx.x / a.tiles;
    const int r = (blockIdx.x - R * a.tiles) * kThreads + threadIdx.x;
    if (r >= a.Z) return;
    const RowDesc rd = tab.row[R];
    const int64_t c = (int64_t)R * a.Z + r;
    float t = 0.0f;
    if (rd.abs_col >= 0) {
        int j = r + rd.abs_shift; j -= (j >= a.Z) ? a.Z : 0;
        t = q_of_llr(__ldg(a.llr + (int64_t)f * a.n + (int64_t)rd.abs_col * a.Z + j));
    }
    const unsigned s = a.syn[(int64_t)f * a.m + c] & 1u;
    a.t[(int64_t)f * a.m + c] = __uint_as_float(__float_as_uint(t) ^ (s << 31));
}

struct CnArgs {
    const float* llr; const uint8_t* syn; const float* qbuf0; const float* qbuf1; uint8_t* hard; float* post;
    const int* done; const int32_t* iters; int* unsat;
    int Z, tiles, t_fixed, count, skip_done; int64_t n, m, EZ;
};

// a3: one thread per check: decision of the absorbed degree-1 variable, parity of the hard decisions against s_c
template <class Tables>
__global__ void __launch_bounds__(kThreads) k_check(const __grid_constant__ Tables tab, const CnArgs a) {
    const int f = blockIdx.y;
    if (a.skip_done && a.done[f]) return;
    const int t = a.t_fixed >= 0 ? a.t_fixed : a.iters[f];  // iteration whose decisions are being formed
    const int R = blockIdx.x / a.tiles;
    const int r = (blockIdx.x - R * a.tiles) * kThreads + threadIdx.x;
    const int Z = a.Z;
    unsigned bad = 0;
    if (r < Z) {
        const RowDesc rd = tab.row[R];
        // m^(t) is formed from the messages of iteration t-1: the buffer k_vn_pass(t) read from
        const float* __restrict__ qprev = (((t - 1) & 1) ? a.qbuf1 : a.qbuf0) + (int64_t)f * a.EZ;
        const uint8_t* hard = a.hard + (int64_t)f * a.n;
        unsigned par = a.syn[(int64_t)f * a.m + (int64_t)R * Z + r] & 1u;
        unsigned sg = par << 31;
        float num = 0.0f, den = 1.0f;
        for (int k = 0; k < rd.ne; ++k) {
            const RowEdge re = tab.redge[rd.ebeg + k];
            int iv = r + re.shift; iv -= (iv >= Z) ? Z : 0;
            par ^= hard[(int64_t)re.col * Z + iv] & 1u;
            if (rd.abs_col >= 0 && t > 0) {
                const float qa = __ldg(qprev + (int64_t)re.edge * Z + iv);
                sg ^= __float_as_uint(qa) & 0x80000000u;
                boxplus_acc(fabsf(qa), num, den);
            }
        }
        if (rd.abs_col >= 0) {
            int j = r + rd.abs_shift; j -= (j >= Z) ? Z : 0;
            const int64_t v = (int64_t)f * a.n + (int64_t)rd.abs_col * Z + j;
            const float Qj = __ldg(a.llr + v);
            const float mcj = t > 0 ? __uint_as_float(__float_as_uint(mag_of(num, den)) | sg) : 0.0f;
            const float Lj = Qj + mcj;                       // degree-1 variable: L_j = Q_j + m_cj
            const unsigned xj = Lj < 0.0f ? 1u : 0u;
            a.hard[v] = (uint8_t)xj;
            if (a.post) a.post[v] = Lj;
            par ^= xj;
        }
        bad = par;
    }
    if (a.count) {
        const int nbad = __syncthreads_count(bad != 0);
        if (threadIdx.x == 0 && nbad) atomicAdd(a.unsat + f, nbad);
    }
}

// a3: per-frame early exit.  mode 0: iteration t of an early-stop run; mode 1: final pass/fail of a fixed-length run
__global__ void k_flags(int* done, int* unsat, int32_t* iters, uint8_t* pass, int n_frames, int t, int final_only) {
    const int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= n_frames) return;
    if (final_only) {
        pass[f] = unsat[f] == 0 ? 1 : 0;
        iters[f] = t;
    } else if (!done[f]) {
        if (unsat[f] == 0) { done[f] = 1; iters[f] = t; pass[f] = 1; }
    }
    unsat[f] = 0;
}

__global__ void k_reset(int* done, int* unsat, int32_t* iters, uint8_t* pass, int n_frames, int max_iter) {
    const int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= n_frames) return;
    done[f] = 0; unsat[f] = 0; iters[f] = max_iter; pass[f] = 0;
}

// ---------------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------------
// kind 0 = k_vn_pass, 1 = k_check.  Returns the pair index to close with prof_end, or -1.
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
    float* qbuf[2]; float* t; int* done; int* unsat;
    size_t bytes;
};

Workspace carve(const qcldpc_code* code, int n_frames, void* base) {
    Workspace w;
    char* p = static_cast<char*>(base);
    size_t off = 0;
    const size_t qbytes = align_up((size_t)n_frames * code->n_act_edges * code->Z * sizeof(float), 256);
    const size_t tbytes = align_up((size_t)n_frames * code->m * sizeof(float), 256);
    const size_t fbytes = align_up((size_t)n_frames * sizeof(int), 256);
    w.qbuf[0] = reinterpret_cast<float*>(p + off); off += qbytes;
    w.qbuf[1] = reinterpret_cast<float*>(p + off); off += qbytes;
    w.t = reinterpret_cast<float*>(p + off); off += tbytes;
    w.done = reinterpret_cast<int*>(p + off); off += fbytes;
    w.unsat = reinterpret_cast<int*>(p + off); off += fbytes;
    w.bytes = off;
    return w;
}

// Register-array size used for a code: the exact degree when every active column has the same degree and a
// specialisation exists (the BASELINE.json codes: 11 and 21), else the next bucket.
int vn_bucket(int max_dv, bool uniform) {
    if (uniform && (max_dv == 11 || max_dv == 21)) return max_dv;
    const int buckets[] = {8, 16, 32, 64};
    for (int b : buckets) if (max_dv <= b) return b;
    return -1;
}
VnLauncher vn_launcher(int bucket) {
    switch (bucket) {
        case 8: return launch_vn_dv8;
        case 11: return launch_vn_dv11;
        case 16: return launch_vn_dv16;
        case 21: return launch_vn_dv21;
        case 32: return launch_vn_dv32;
        case 64: return launch_vn_dv64;
        default: return nullptr;
    }
}

void launch_check(const qcldpc_code* code, const CnArgs& a, dim3 grid, cudaStream_t st) {
    if (code->inline_ok) k_check<CnTablesInline><<<grid, kThreads, 0, st>>>(code->cn_inl, a);
    else k_check<CnTablesGlobal><<<grid, kThreads, 0, st>>>(CnTablesGlobal{code->d_row, code->d_redge}, a);
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------------
// C ABI
// ---------------------------------------------------------------------------------------------------------------
extern "C" {

int qcldpc_code_create(const int32_t* base, int mb, int nb, int Z, qcldpc_code_t** out_code) {
    if (!base || !out_code || mb <= 0 || nb <= 0 || Z <= 0) return QCLDPC_ERR_BAD_ARGUMENT;
    *out_code = nullptr;
    if ((int64_t)mb * Z > (int64_t)1 << 30 || (int64_t)nb * Z > (int64_t)1 << 30) return QCLDPC_ERR_UNSUPPORTED;
    for (int64_t k = 0; k < (int64_t)mb * nb; ++k)
        if (base[k] < -1 || base[k] >= Z) return QCLDPC_ERR_BAD_ARGUMENT;
    qcldpc_code* code = new (std::nothrow) qcldpc_code();
    if (!code) return QCLDPC_ERR_ALLOC;
    code->mb = mb; code->nb = nb; code->Z = Z;
    code->n = (int64_t)nb * Z; code->m = (int64_t)mb * Z;

    // column degrees; absorb at most one degree-1 column per row (the lowest-numbered one)
    std::vector<int> deg(nb, 0), absorbed_by(nb, -1);
    for (int R = 0; R < mb; ++R)
        for (int C = 0; C < nb; ++C) deg[C] += base[(size_t)R * nb + C] >= 0;
    code->row.assign(mb, RowDesc{0, 0, -1, 0});
    for (int R = 0; R < mb; ++R)
        for (int C = 0; C < nb; ++C)
            if (base[(size_t)R * nb + C] >= 0 && deg[C] == 1 && code->row[R].abs_col < 0) {
                code->row[R].abs_col = C;
                code->row[R].abs_shift = base[(size_t)R * nb + C];
                absorbed_by[C] = R;
            }
    // active columns and their edges, in increasing (column, row) order
    struct HostEdge { int shift, row, col_k; };
    std::vector<HostEdge> edges;
    std::vector<int> edge_of_cell((size_t)mb * nb, -1);
    code->max_dv = 0;
    bool uniform = true;
    int first_dv = -1;
    for (int C = 0; C < nb; ++C) {
        if (absorbed_by[C] >= 0) continue;
        ColDesc cd{C, (int)edges.size(), 0, 0, 0, 0, 0, 0};
        for (int R = 0; R < mb; ++R) {
            const int p = base[(size_t)R * nb + C];
            if (p < 0) continue;
            edge_of_cell[(size_t)R * nb + C] = (int)edges.size();
            edges.push_back(HostEdge{p, R, cd.dv});
            ++cd.dv;
        }
        code->col.push_back(cd);
        code->max_dv = std::max(code->max_dv, cd.dv);
        if (first_dv < 0) first_dv = cd.dv;
        uniform = uniform && cd.dv == first_dv;
    }
    code->n_act_cols = (int)code->col.size();
    code->n_act_edges = (int)edges.size();
    if (code->max_dv > kMaxDv || (int64_t)code->n_act_edges * Z >= ((int64_t)1 << 31)) {
        delete code;
        return QCLDPC_ERR_UNSUPPORTED;
    }
    // row view
    for (int R = 0; R < mb; ++R) {
        code->row[R].ebeg = (int)code->redge.size();
        for (int C = 0; C < nb; ++C) {
            const int e = edge_of_cell[(size_t)R * nb + C];
            if (e >= 0) code->redge.push_back(RowEdge{e, base[(size_t)R * nb + C], C, 0});
        }
        code->row[R].ne = (int)code->redge.size() - code->row[R].ebeg;
    }
    // per edge: the pair descriptor; rows with 0 or >= 2 other active edges get a partner list (GenDesc)
    for (size_t ci = 0; ci < code->col.size(); ++ci) {
        ColDesc& cd = code->col[ci];
        cd.gbeg = (int)code->gen.size();
        for (int k = 0; k < cd.dv; ++k) {
            const int e = cd.ebeg + k;
            const HostEdge& he = edges[e];
            const RowDesc& rd = code->row[he.row];
            PairDesc pd{he.shift, he.row * Z, -1, 0};
            const int np = rd.ne - 1;
            if (np == 1) {
                for (int j = 0; j < rd.ne; ++j) {
                    const RowEdge& re = code->redge[rd.ebeg + j];
                    if (re.edge == e) continue;
                    pd.p_off = re.edge * Z;
                    pd.delta = ((re.shift - he.shift) % Z + Z) % Z;
                }
            } else {
                GenDesc gd{k, (int)code->partner.size(), np, 0};
                for (int j = 0; j < rd.ne; ++j) {
                    const RowEdge& re = code->redge[rd.ebeg + j];
                    if (re.edge == e) continue;
                    code->partner.push_back(PartnerDesc{re.edge * Z, ((re.shift - he.shift) % Z + Z) % Z});
                }
                code->gen.push_back(gd);
            }
            code->pair.push_back(pd);
        }
        cd.ng = (int)code->gen.size() - cd.gbeg;
    }
    code->n_partners = (int)code->partner.size();
    code->uniform_dv = uniform && code->n_act_cols > 0;
    code->bucket = vn_bucket(code->max_dv, code->uniform_dv);
    code->launcher = vn_launcher(code->bucket);
    code->inline_ok = code->n_act_edges <= kInlEdges && code->n_partners <= kInlPartners &&
                      code->n_act_cols <= kInlCols && (int)code->gen.size() <= kInlGen && mb <= kInlRows;
    if (code->inline_ok) {
        memset(&code->vn_inl, 0, sizeof(code->vn_inl));
        memset(&code->cn_inl, 0, sizeof(code->cn_inl));
        std::copy(code->pair.begin(), code->pair.end(), code->vn_inl.pair);
        std::copy(code->partner.begin(), code->partner.end(), code->vn_inl.partner);
        std::copy(code->gen.begin(), code->gen.end(), code->vn_inl.gen);
        std::copy(code->col.begin(), code->col.end(), code->vn_inl.col);
        std::copy(code->row.begin(), code->row.end(), code->cn_inl.row);
        std::copy(code->redge.begin(), code->redge.end(), code->cn_inl.redge);
    }
    // device copies (always made: the init kernels and large codes read them from global memory)
    auto upload = [](auto& vec, auto** dptr) -> cudaError_t {
        const size_t bytes = std::max<size_t>(vec.size(), 1) * sizeof(vec[0]);
        cudaError_t e = cudaMalloc(reinterpret_cast<void**>(dptr), bytes);
        if (e != cudaSuccess) return e;
        if (!vec.empty()) e = cudaMemcpy(*dptr, vec.data(), vec.size() * sizeof(vec[0]), cudaMemcpyHostToDevice);
        return e;
    };
    cudaError_t e = upload(code->pair, &code->d_pair);
    if (e == cudaSuccess) e = upload(code->partner, &code->d_partner);
    if (e == cudaSuccess) e = upload(code->gen, &code->d_gen);
    if (e == cudaSuccess) e = upload(code->col, &code->d_col);
    if (e == cudaSuccess) e = upload(code->row, &code->d_row);
    if (e == cudaSuccess) e = upload(code->redge, &code->d_redge);
    if (e != cudaSuccess) { qcldpc_code_destroy(code); return cuda_fail(e, "qcldpc_code_create: table upload"); }
    *out_code = code;
    return QCLDPC_OK;
}

void qcldpc_code_destroy(qcldpc_code_t* code) {
    if (!code) return;
    cudaFree(code->d_pair); cudaFree(code->d_partner); cudaFree(code->d_gen); cudaFree(code->d_col);
    cudaFree(code->d_row); cudaFree(code->d_redge);
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
    g_launches = 0;
    if (!code || !d_llr || !d_syndrome || !d_hard || !d_iters || !d_pass) return QCLDPC_ERR_BAD_ARGUMENT;
    if (n_frames <= 0 || n_frames > 65535 || max_iter < 0) return QCLDPC_ERR_BAD_ARGUMENT;
    if (!d_workspace || (reinterpret_cast<uintptr_t>(d_workspace) & 255) ||
        workspace_bytes < qcldpc_workspace_bytes(code, n_frames))
        return QCLDPC_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const Workspace w = carve(code, n_frames, d_workspace);
    const int Z = code->Z;
    const int64_t EZ = (int64_t)code->n_act_edges * Z;
    const int tiles1 = (Z + kThreads - 1) / kThreads;
    const int fblocks = (n_frames + 127) / 128;

    k_reset<<<fblocks, 128, 0, st>>>(w.done, w.unsat, d_iters, d_pass, n_frames, max_iter);
    ++g_launches;
    InitArgs ia{d_llr, d_syndrome, w.qbuf[0], w.t, d_hard, d_posterior, Z, tiles1, code->n, code->m, EZ};
    if (code->n_act_cols > 0) {
        k_init_q<VnTablesGlobal><<<dim3(tiles1 * code->n_act_cols, n_frames), kThreads, 0, st>>>(
            VnTablesGlobal{code->d_pair, code->d_partner, code->d_gen, code->d_col}, ia);
        ++g_launches;
    }
    k_init_t<CnTablesGlobal><<<dim3(tiles1 * code->mb, n_frames), kThreads, 0, st>>>(
        CnTablesGlobal{code->d_row, code->d_redge}, ia);
    ++g_launches;

    const dim3 grid_vn(tiles1 * code->n_act_cols, n_frames);
    if (code->n_act_cols > 0 && !code->launcher) return QCLDPC_ERR_UNSUPPORTED;
    const dim3 grid_cn(tiles1 * code->mb, n_frames);
    CnArgs ca{d_llr, d_syndrome, w.qbuf[0], w.qbuf[1], d_hard, nullptr, w.done, d_iters, w.unsat,
              Z, tiles1, 0, 1, 1, code->n, code->m, EZ};

    for (int t = 1; t <= max_iter; ++t) {
        if (code->n_act_cols > 0) {
            VnLaunch vl{code->inline_ok ? &code->vn_inl : nullptr,
                        VnTablesGlobal{code->d_pair, code->d_partner, code->d_gen, code->d_col},
                        VnArgs{d_llr, w.qbuf[(t - 1) & 1], w.qbuf[t & 1], w.t, d_hard, d_posterior, w.done,
                               Z, tiles1, code->n, code->m, EZ},
                        grid_vn, st};
            const int pk = prof_begin(0, st);
            code->launcher(vl);
            prof_end(pk, st);
            ++g_launches;
        }
        if (early_stop) {
            ca.t_fixed = t;
            const int pk = prof_begin(1, st);
            launch_check(code, ca, grid_cn, st);
            prof_end(pk, st);
            k_flags<<<fblocks, 128, 0, st>>>(w.done, w.unsat, d_iters, d_pass, n_frames, t, 0);
            g_launches += 2;
        }
    }
    if (!early_stop || max_iter == 0) {
        // fixed-length run: one check of the final decisions gives d_pass (and the absorbed variables' outputs)
        ca.t_fixed = max_iter; ca.post = d_posterior; ca.skip_done = 0;
        launch_check(code, ca, grid_cn, st);
        k_flags<<<fblocks, 128, 0, st>>>(w.done, w.unsat, d_iters, d_pass, n_frames, max_iter, 1);
        g_launches += 2;
    } else if (d_posterior) {
        // early-stop run: posteriors of the absorbed variables from each frame's frozen state (iteration d_iters[f])
        ca.t_fixed = -1; ca.post = d_posterior; ca.skip_done = 0; ca.count = 0;
        launch_check(code, ca, grid_cn, st);
        ++g_launches;
    }
    CUDA_TRY(cudaGetLastError());
    return QCLDPC_OK;
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
    g_launches = 0;
    if (!code || !h_llr || !h_syndrome || !h_hard || !h_iters || !h_pass) return QCLDPC_ERR_BAD_ARGUMENT;
    if (n_frames <= 0 || max_iter < 0) return QCLDPC_ERR_BAD_ARGUMENT;
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
    const int rc = qcldpc_decode(code, d_llr, d_syn, n_frames, max_iter, early_stop, d_hard, d_iters, d_pass, d_post,
                                 d_workspace, core, stream);
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
        case QCLDPC_ERR_UNSUPPORTED: return "unsupported code (active column degree > 64 or size out of range)";
        case QCLDPC_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
        case QCLDPC_ERR_CUDA: return "CUDA runtime error";
        case QCLDPC_ERR_ALLOC: return "host allocation failed";
        default: return "unknown status";
    }
}

const char* qcldpc_last_cuda_error(void) { return g_cuda_error; }

}  // extern "C"

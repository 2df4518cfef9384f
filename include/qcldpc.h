/*
 * qcldpc.h -- C ABI of libqcldpc: B200 (sm_100a) flooding Sum-Product decoder for quasi-cyclic LDPC codes in
 * syndrome form (the decoder gets channel LLRs and a syndrome s and must reach H xhat = s).
 *
 * What is computed (citations: /root/reference/PAPER.md line numbers, "P:NNN"; readings S1..S14 in DESIGN.md):
 *   Algorithm 1 of the paper: LLR initialisation L_vc <- Q_v; per iteration the check-node update
 *   sgn(m_cv) = (-1)^{s_c} prod_{v' in N(c)\v} sgn(L_v'c),  |m_cv| = Phi^-1( sum_{v' in N(c)\v} Phi(|L_v'c|) ),
 *   Phi(x) = -ln tanh(x/2) (the factor (-1)^{s_c} is the syndrome generalisation, S1),
 *   clamped to |m_cv| <= QCLDPC_MSG_MAX (S2); the variable-node update L_vc = Q_v + sum_{c' in M(v)\c} m_c'v and
 *   posterior L_v = Q_v + sum_{c in M(v)} m_cv; the hard decision xhat_v = 0 iff L_v >= 0 and
 *   the early-termination test H xhat = s (mod 2) (P:363 generalised), per frame.
 *   H is given as a base matrix of circulant shifts and a lifting size Z.
 *
 * All computation runs in CUDA kernels on the current device; there is no CPU fallback.  No function throws or
 * exits; every function returns a status (0 = success, negative = error, see qcldpc_status_string).
 */
#ifndef QCLDPC_H_
#define QCLDPC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define QCLDPC_MSG_MAX 30.0f /* clamp on |m_cv| (reading S2); part of the definition of the result */
#define QCLDPC_MAX_FRAMES 65535 /* frames per decode call (one grid dimension of the kernels); more: split the batch */
#define QCLDPC_STATIC_WORKSPACE_BYTES (16u << 20) /* the library's own workspace of qcldpc_decode_static: 16 MiB per GPU */

enum {
    QCLDPC_OK = 0,
    QCLDPC_ERR_BAD_ARGUMENT = -1, /* NULL pointer, non-positive size, shift outside [-1, Z), max_iter < 0, ... */
    QCLDPC_ERR_UNSUPPORTED = -2,  /* code outside the supported envelope, see qcldpc_code_create */
    QCLDPC_ERR_WORKSPACE = -3,    /* workspace NULL, misaligned (256 B) or smaller than qcldpc_workspace_bytes */
    QCLDPC_ERR_CUDA = -4,         /* a CUDA runtime call failed; qcldpc_last_cuda_error() has the text */
    QCLDPC_ERR_ALLOC = -5         /* host allocation failed */
};

typedef struct qcldpc_code qcldpc_code_t;

/*
 * Build a code handle from a base matrix.
 *   base_shifts  HOST pointer, int32 row-major [mb][nb]; -1 = all-zero ZxZ block; p in [0,Z) = the ZxZ identity with
 *                every row cyclically shifted right by p (the paper's entry i = p+1, I_i): check R*Z + r is connected
 *                to variable C*Z + ((r + p) mod Z).  Rows are checks, columns are variables.
 *   mb, nb, Z    > 0.   n = nb*Z variables, m = mb*Z checks.
 *   out_code     receives the handle (owned by the caller, release with qcldpc_code_destroy).
 * The handle owns small device tables (allocated with cudaMalloc on the current device) and is immutable: it may be
 * used concurrently from several streams with distinct workspaces.  At most one degree-1 column per base row is
 * "absorbed" into that row (such variables send Q_v forever and need no edge state); every other column is
 * "active" and carries one fp32 of state per edge.
 * Supported envelope (else QCLDPC_ERR_UNSUPPORTED): active columns of degree 0..64; at most 2048 partner entries per
 * active column (the sum, over the column's edges into rows that are not "two active edges + one absorbed variable",
 * of that row's other active edges); mb*Z and nb*Z at most 2^30; a frame's edge state (active base edges x Z rounded up
 * to a multiple of 8, or Z + 256 rounded up to 32 for the BASELINE.json column shapes) and mb x that run length each
 * below 2^30 floats (the kernels form 32-bit byte offsets inside a frame).
 * Tuning knobs: qcldpc_code_create reads these environment variables ONCE and stores them in the handle; no decode
 * call reads the environment.  Defaults are the measured best.  QCLDPC_V=1|2 variables per thread
 * of the exact pass; QCLDPC_FLIP=0 every launch walks the frames forwards; QCLDPC_MERGE_CHECK=0 early-exit check as a
 * separate launch; QCLDPC_CAND_PER_SM=k grid of that launch; QCLDPC_PACK=0 no lane packing and QCLDPC_FV=1|2 frames
 * per thread in the generic pass; QCLDPC_LOOP=stream and QCLDPC_BODY=k (body of 12 k iterations) for the iteration
 * loop (see qcldpc_iterations_issued); QCLDPC_IL=0|2 never / always the frame-interleaved kernel family, QCLDPC_ILW=k
 * its variables per CTA, QCLDPC_ILA=0..4 the depth of its asynchronous pipeline in chunks of four edges (0: loads
 * through registers and messages in shared memory; default 2: messages in tensor memory, for columns of more than 16
 * edges).  None of them changes any result.
 */
int qcldpc_code_create(const int32_t* base_shifts, int mb, int nb, int Z, qcldpc_code_t** out_code);
void qcldpc_code_destroy(qcldpc_code_t* code);

/*
 * The same handle from the NON-ZERO blocks only (for large base graphs, e.g. the paper's own ensemble with ~20,000
 * base columns and q = 50, whose dense [mb][nb] array would be 1.5 GB):
 *   rows, cols, shifts  HOST pointers, int32 [n_entries]: block (rows[k], cols[k]) is the identity shifted right by
 *                       shifts[k] in [0,Z); any order; every other block is zero.  A repeated (row, col) pair is an
 *                       error (a block is one circulant).
 * qcldpc_code_create(base, ...) equals qcldpc_code_create_sparse of the cells of base that are >= 0.
 */
int qcldpc_code_create_sparse(const int32_t* rows, const int32_t* cols, const int32_t* shifts, int64_t n_entries,
                              int mb, int nb, int Z, qcldpc_code_t** out_code);

/* Code facts: n, m, number of active base edges (one fp32 of state per active edge and buffer; four buffers). */
int qcldpc_code_info(const qcldpc_code_t* code, int64_t* n, int64_t* m, int64_t* active_base_edges);

/* Bytes of DEVICE workspace qcldpc_decode needs for n_frames frames (0 on bad arguments). */
size_t qcldpc_workspace_bytes(const qcldpc_code_t* code, int n_frames);

/*
 * Decode n_frames independent frames (Algorithm 1, syndrome form), 1 <= n_frames <= QCLDPC_MAX_FRAMES.
 * Only ENQUEUES work on `stream`; never synchronises the device; allocates no device memory of its own (the first call
 * of a process on a device sets kernel attributes; the first call with a new argument tuple instantiates a CUDA graph,
 * see qcldpc_iterations_issued).  All d_* are DEVICE pointers owned by the caller, frame-major and
 * contiguous:
 *   d_llr        const float   [n_frames][n]  Q_v = ln P(x_v=0)/P(x_v=1)
 *   d_syndrome   const uint8_t [n_frames][m]  s_c in {0,1} (only bit 0 is read)
 *   max_iter     >= 0.  max_iter = 0: xhat = [Q < 0], d_iters = 0, d_pass by direct check (S6)
 *   early_stop   0: exactly max_iter iterations, d_iters[f] = max_iter;  1: frame f stops at the first iteration t
 *                (1-based) with H xhat = s, its outputs are those of iteration t (S5-S7)
 *   d_hard       uint8_t [n_frames][n]   xhat_v = (L_v < 0) of the frame's last executed iteration
 *   d_iters      int32_t [n_frames]      iteration at which the frame stopped, else max_iter
 *   d_pass       uint8_t [n_frames]      1 iff H d_hard = d_syndrome
 *   d_posterior  float   [n_frames][n]   L_v of the frame's last executed iteration; may be NULL
 *   d_workspace  >= qcldpc_workspace_bytes(code, n_frames) bytes, 256-byte aligned; contents are scratch
 *   stream       cudaStream_t passed as void* (NULL = the legacy default stream)
 * Returns QCLDPC_OK once everything is enqueued.  Outputs are valid when the stream has drained.
 */
int qcldpc_decode(const qcldpc_code_t* code, const float* d_llr, const uint8_t* d_syndrome, int n_frames,
                  int max_iter, int early_stop, uint8_t* d_hard, int32_t* d_iters, uint8_t* d_pass,
                  float* d_posterior, void* d_workspace, size_t workspace_bytes, void* stream);

/*
 * qcldpc_decode with the paper's early-termination scheduling (the parity test is "enabled only after"
 * an expected number of iterations, which the paper takes from a per-SNR table of average iteration counts):
 *   check_from_iter  >= 1.  With early_stop = 1 the test H xhat = s runs at iterations t >= check_from_iter only; a
 *                    frame cannot stop earlier, d_iters[f] >= check_from_iter for every frame that stops.
 *                    check_from_iter = 1 is qcldpc_decode (test at every iteration, reading S5).  No effect when
 *                    early_stop = 0.  The caller supplies the number (the paper's table is not published).
 * Everything else as qcldpc_decode.  Before check_from_iter the per-iteration early-exit kernel is not launched.
 */
int qcldpc_decode_ex(const qcldpc_code_t* code, const float* d_llr, const uint8_t* d_syndrome, int n_frames,
                     int max_iter, int early_stop, int check_from_iter, uint8_t* d_hard, int32_t* d_iters,
                     uint8_t* d_pass, float* d_posterior, void* d_workspace, size_t workspace_bytes, void* stream);

/*
 * Same decode with HOST buffers (h_* are HOST pointers, same shapes; pinned memory makes the copies asynchronous):
 * copies inputs host->device, decodes, copies outputs device->host on `stream`, then WAITS for the stream so that the
 * h_* outputs are valid on return.  The iteration loop ends on the device as in qcldpc_decode (with QCLDPC_LOOP=stream
 * this call reads the number of live frames back every 32 iterations and stops launching once every frame has stopped).
 * h_posterior may be NULL.  The device staging area is part of d_workspace, which
 * must hold qcldpc_host_workspace_bytes(code, n_frames, h_posterior != NULL) bytes.
 */
size_t qcldpc_host_workspace_bytes(const qcldpc_code_t* code, int n_frames, int want_posterior);
int qcldpc_decode_host(const qcldpc_code_t* code, const float* h_llr, const uint8_t* h_syndrome, int n_frames,
                       int max_iter, int early_stop, uint8_t* h_hard, int32_t* h_iters, uint8_t* h_pass,
                       float* h_posterior, void* d_workspace, size_t workspace_bytes, void* stream);
/* qcldpc_decode_host with the early-termination scheduling of qcldpc_decode_ex (check_from_iter >= 1). */
int qcldpc_decode_host_ex(const qcldpc_code_t* code, const float* h_llr, const uint8_t* h_syndrome, int n_frames,
                          int max_iter, int early_stop, int check_from_iter, uint8_t* h_hard, int32_t* h_iters,
                          uint8_t* h_pass, float* h_posterior, void* d_workspace, size_t workspace_bytes,
                          void* stream);

/*
 * ---- The steps either side of the decoder (device pointers; each call only enqueues on `stream`) ----
 *
 * LLR front end, Step 1 of Algorithm 1: sigma^2_{N_v} <- sigma^2_Z / ||X_v||, Q_v <- 2 R_v / sigma^2_{N_v}.
 *   d_r, d_x     const float [n_frames][n]  Alice's received values R_v = M_v / X_v (Eq. 1) and her own X_v
 *   d_sigma2_z   const float [n_frames]     channel noise variance sigma^2_Z of each frame
 *   dim          0: no side information, sigma^2_N = sigma^2_Z for every symbol (d_x may be NULL; this is the BIAWGN
 *                   recipe LLR = 2 y / sigma^2 of BASELINE.json's configs)
 *                1: the d = 1 scheme: sigma^2_{N_v} = sigma^2_Z / ||X_v||^norm_power.  norm_power = 2 is the
 *                   variance Eq. 1 implies (noise term Z_v / X_v) and the one under which Q_v is the log-likelihood
 *                   ratio Step 1 says it is; norm_power = 1 is the formula as printed at P:97 / P:344 (reading G5)
 *                2: the d = 2 scheme: successive pairs (2i, 2i+1), 0-based, n even:
 *                   a = (X_2i + X_2i+1) / (X_2i^2 + X_2i+1^2), b = (X_2i+1 - X_2i) / (same), sigma^2_N = (a^2 + b^2) sigma^2_Z
 *                   (the d = 4 and d = 8 noise terms are not in the paper)
 *   d_llr        float [n_frames][n]        Q_v, the input of qcldpc_decode
 * IEEE single-precision arithmetic in the printed order (X_v = 0: infinite variance, Q_v = +-0).
 */
int qcldpc_llr_init(const float* d_r, const float* d_x, const float* d_sigma2_z, int n_frames, int64_t n, int dim,
                    int norm_power, float* d_llr, void* stream);

/*
 * Bit-packed outputs (Step 5, keeps the first k bits of the decoded word): the first n_bits <= n hard decisions
 * of every frame of d_hard (uint8 [n_frames][n], one byte per bit, only bit 0 is read) as (n_bits + 7) / 8 bytes per
 * frame in d_packed (uint8 [n_frames][(n_bits + 7) / 8]); bit v of a frame is bit 7 - (v mod 8) of byte v / 8 (most
 * significant bit first, reading G8); unused low bits of the last byte are zero.
 */
int qcldpc_pack_bits(const uint8_t* d_hard, int n_frames, int64_t n, int64_t n_bits, uint8_t* d_packed, void* stream);

/*
 * 32-bit CRC of each decoded message against the CRC that travels in the frame (Fig. 7: the k information
 * bits are k - 32 message bits followed by N_CRC = 32 CRC bits; run it on the frames whose parity check
 * passed).  CRC-32 of IEEE 802.3 (reading G7: polynomial 0x04C11DB7 bit-reflected, initial value and final XOR
 * 0xFFFFFFFF; "123456789" -> 0xCBF43926) over the first (k_bits - 32) / 8 bytes of every row of d_packed; the stored
 * CRC is the big-endian 32-bit number in the next 4 bytes.
 *   d_packed      const uint8_t [n_frames][stride_bytes], stride_bytes >= k_bits / 8 (qcldpc_pack_bits output)
 *   k_bits        a multiple of 8, >= 32
 *   d_crc         uint32_t [n_frames]  the computed CRC (may be NULL)
 *   d_ok          uint8_t  [n_frames]  1 iff computed == stored (may be NULL; not both NULL)
 */
int qcldpc_crc32_check(const uint8_t* d_packed, int n_frames, int64_t stride_bytes, int64_t k_bits, uint32_t* d_crc,
                       uint8_t* d_ok, void* stream);

/* Number of kernel launches (graph path: kernel nodes, the loop body counted once) the last qcldpc_decode /
 * qcldpc_decode_host call of this thread enqueued. */
int64_t qcldpc_last_launch_count(void);

/*
 * The iteration loop runs on the DEVICE: by default a decode call builds (first call with a given argument tuple) and
 * launches ONE CUDA graph whose conditional WHILE node repeats a body of 12 iterations until max_iter is reached or
 * every frame of the batch has stopped ("Go to Step 5"), so a batch that has stopped costs at most one more body
 * of empty launches although the call never waits.  Instantiated graphs are cached in the handle, keyed by all pointer
 * and scalar arguments (the one place where the handle changes after creation; guarded by a mutex; building a graph
 * allocates driver memory).  QCLDPC_LOOP=stream (read by qcldpc_code_create) keeps one launch per iteration from the
 * host; so do decodes of fewer than 14 iterations, calls made while qcldpc_profile_enable is on, and calls on a stream
 * that the caller is capturing into a graph of its own (the launches then become nodes of that graph).
 *   qcldpc_iterations_issued  how many iterations' launches the last decode in d_workspace actually issued (reads one
 *                             int back from the workspace on `stream` and WAITS for it; h_iterations: HOST pointer)
 *   qcldpc_last_loop_mode     1 if the last decode call of this thread ran as a graph, 0 if as stream launches
 */
int qcldpc_iterations_issued(const qcldpc_code_t* code, int n_frames, const void* d_workspace, void* stream,
                             int* h_iterations);
int qcldpc_last_loop_mode(void);

/*
 * qcldpc_decode_static: qcldpc_decode_ex for callers that cannot allocate device memory (code under CUDA graph capture,
 * serving loops, harnesses that forbid cudaMalloc).  Same operation (Algorithm 1, syndrome form), same
 * arguments, layouts and outputs as qcldpc_decode_ex, but NO workspace argument: the decoder's scratch memory (four
 * buffers of edge state, the static check terms, the decisions, the per-frame flags) lives in a device array of
 * QCLDPC_STATIC_WORKSPACE_BYTES = 16 MiB that is part of the library image: every GPU that loads the library holds it
 * until the process exits.  The call itself calls no cudaMalloc / cudaFree and no allocating library routine: it only
 * enqueues plain kernel launches on `stream`, one pass per iteration for all max_iter iterations (no device-side graph
 * loop -- building a graph allocates --, no host polling, never waits); on a stream the caller is capturing the
 * launches become nodes of the caller's graph.  The code handle (whose tables qcldpc_code_create allocates) must exist.
 *   Limit: qcldpc_workspace_bytes(code, n_frames) <= qcldpc_static_workspace_bytes(), else QCLDPC_ERR_WORKSPACE with
 *   the two sizes in qcldpc_last_cuda_error() (BASELINE.json's config 1 fits with up to about 90 frames; the n = 10^6
 *   codes do not: they take qcldpc_decode with a workspace of the caller's).  QCLDPC_ERR_BAD_ARGUMENT while
 *   qcldpc_profile_enable is on (the profile allocates events), other errors as qcldpc_decode_ex.
 *   Sharing: every call on a GPU uses the SAME array, which keeps the previous call's contents; each call first clears
 *   and rewrites all of it that it reads.  Two calls that overlap on the GPU (different streams, or replays of two
 *   captured graphs at once) race on it: serialise them on one stream or with events.  One array per GPU: calls on
 *   different GPUs are independent.
 * qcldpc_static_workspace_bytes: the size of that array.
 */
int qcldpc_decode_static(const qcldpc_code_t* code, const float* d_llr, const uint8_t* d_syndrome, int n_frames,
                         int max_iter, int early_stop, int check_from_iter, uint8_t* d_hard, int32_t* d_iters,
                         uint8_t* d_pass, float* d_posterior, void* stream);
size_t qcldpc_static_workspace_bytes(void);

const char* qcldpc_status_string(int status);
const char* qcldpc_last_cuda_error(void); /* thread-local text of the last CUDA failure ("" if none) */

#ifdef __cplusplus
}
#endif
#endif /* QCLDPC_H_ */

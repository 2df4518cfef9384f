// l2_path_probe -- stand-alone measurement tool (not part of libqcldpc): throughput of the fused pass's ACCESS PATTERN
// without its arithmetic.  Per CTA: R read streams of `tile` consecutive floats at arbitrary (unaligned) cyclic shifts
// inside runs of Zs floats, W aligned write streams, for 64 frames x 10 columns x Z = 10000 like config 4.  DUP of the R
// read streams re-read another column's data (served from L2, like t_c and the gen-row states in k_pass).  Prints the
// DRAM-level GB/s (unique bytes / time).  Used for DESIGN.md §5 "what actually caps it"; results in
// profiles/r01c_l2_path.md.
//   nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o l2_path_probe paper_1702_07740_b200/csrc/l2_path_probe.cu
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdlib>
#include <vector>

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { printf("%s: %s\n", #x, cudaGetErrorString(e_)); exit(1); } } while (0)

struct Args { const int* done; const float* in; float* out; const int* shifts; int Z, Zs, R, W, cols; long long in_frame, out_frame; };

template <int THREADS, int V, int R, int W, int DUP, int GATE>
__global__ void __launch_bounds__(THREADS) k_streams(Args a) {
    if (GATE && a.done[blockIdx.z]) return;
    const int f = blockIdx.z, c = blockIdx.y;
    const int i0 = blockIdx.x * THREADS * V;
    const int tid = threadIdx.x;
    constexpr int RU = R - DUP;
    const float* in = a.in + f * a.in_frame + (long long)c * RU * a.Zs;
    const float* in2 = a.in + f * a.in_frame + (long long)((c + 1) % a.cols) * RU * a.Zs;
    float acc[V];
#pragma unroll
    for (int v = 0; v < V; ++v) acc[v] = 0.f;
    float val[R][V];
#pragma unroll
    for (int k = 0; k < R; ++k) {
        int x = i0 + a.shifts[c * R + k]; x -= (x >= a.Z) ? a.Z : 0;
#pragma unroll
        for (int v = 0; v < V; ++v) val[k][v] = __ldg((k < RU ? in + (long long)k * a.Zs : in2 + (long long)(k - RU) * a.Zs) + x + v * THREADS + tid);
    }
#pragma unroll
    for (int k = 0; k < R; ++k)
#pragma unroll
        for (int v = 0; v < V; ++v) acc[v] += val[k][v];
    float* out = a.out + f * a.out_frame + (long long)c * W * a.Zs + i0 + tid;
#pragma unroll
    for (int k = 0; k < W; ++k)
#pragma unroll
        for (int v = 0; v < V; ++v)
            if (i0 + v * THREADS + tid < a.Z) out[(long long)k * a.Zs + v * THREADS] = acc[v] + k;
}

template <int THREADS, int V, int R, int W, int DUP = 0, int GATE = 0>
void run(const char* name, int align, int F, int cols, int Z) {
    const int tile = THREADS * V;
    const int Zs = (Z + 2048 + 31) / 32 * 32;
    Args a;
    a.Z = Z; a.Zs = Zs; a.R = R; a.W = W; a.cols = cols;
    a.in_frame = (long long)cols * (R - DUP) * Zs; a.out_frame = (long long)cols * W * Zs;
    float *in, *out; int* sh;
    CK(cudaMalloc(&in, sizeof(float) * a.in_frame * F));
    CK(cudaMalloc(&out, sizeof(float) * a.out_frame * F));
    CK(cudaMemset(in, 0, sizeof(float) * a.in_frame * F));
    std::vector<int> hs(cols * R);
    srand(1);
    for (auto& s : hs) { s = rand() % Z; if (align) s = s / align * align; }
    CK(cudaMalloc(&sh, sizeof(int) * hs.size()));
    CK(cudaMemcpy(sh, hs.data(), sizeof(int) * hs.size(), cudaMemcpyHostToDevice));
    int* done; CK(cudaMalloc(&done, 4 * F)); CK(cudaMemset(done, 0, 4 * F)); a.done = done;
    a.in = in; a.out = out; a.shifts = sh;
    dim3 grid((Z + tile - 1) / tile, cols, F);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    for (int i = 0; i < 3; ++i) k_streams<THREADS, V, R, W, DUP, GATE><<<grid, THREADS>>>(a);
    CK(cudaDeviceSynchronize());
    const int reps = 20;
    cudaEventRecord(e0);
    for (int i = 0; i < reps; ++i) k_streams<THREADS, V, R, W, DUP, GATE><<<grid, THREADS>>>(a);
    cudaEventRecord(e1);
    CK(cudaDeviceSynchronize());
    float ms; cudaEventElapsedTime(&ms, e0, e1); ms /= reps;
    const double bytes = 4.0 * (R - DUP + W) * (double)Z * cols * F;
    int nb = 0; cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_streams<THREADS, V, R, W, DUP, GATE>, THREADS, 0);
    printf("%-28s align=%-3d DUP=%d GATE=%d R=%d W=%d tile=%4d blocks/SM=%d  %.4f ms  %.0f GB/s\n", name, align, DUP, GATE, R, W, tile, nb, ms, bytes / ms / 1e6);
    cudaFree(in); cudaFree(out); cudaFree(sh);
}

__global__ void k_copy(const float4* __restrict__ a, float4* __restrict__ b, long long n) {
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) b[i] = a[i];
}

int main() {
    const int F = 64, cols = 10, Z = 10000;
    {   // plain copy reference
        long long n = 1ll << 27;   // float4 elements: 2 GiB each
        float4 *a, *b; CK(cudaMalloc(&a, n * 16)); CK(cudaMalloc(&b, n * 16)); CK(cudaMemset(a, 0, n * 16));
        cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
        for (int i = 0; i < 2; ++i) k_copy<<<(unsigned)(n / 256), 256>>>(a, b, n);
        cudaEventRecord(e0);
        for (int i = 0; i < 5; ++i) k_copy<<<(unsigned)(n / 256), 256>>>(a, b, n);
        cudaEventRecord(e1); CK(cudaDeviceSynchronize());
        float ms; cudaEventElapsedTime(&ms, e0, e1); ms /= 5;
        printf("copy float4 2GiB: %.3f ms %.0f GB/s\n", ms, 2.0 * n * 16 / ms / 1e6);
        cudaFree(a); cudaFree(b);
    }
    run<128, 1, 33, 21>("t128 v1 unique streams", 0, F, cols, Z);
    run<128, 1, 33, 21>("t128 v1 unique, aligned", 32, F, cols, Z);
    run<128, 2, 33, 21>("t128 v2 unique streams", 0, F, cols, Z);
    run<256, 2, 33, 21>("t256 v2 unique streams", 0, F, cols, Z);
    run<128, 1, 54, 21>("t128 v1 R54 unique", 0, F, cols, Z);
    run<128, 1, 44, 21, 11>("t128 v1 11 of 44 from L2", 0, F, cols, Z);
    run<128, 1, 54, 21, 21>("t128 v1 21 of 54 from L2", 0, F, cols, Z);
    run<128, 1, 54, 21, 21>("t128 v1 21 of 54 L2, aligned", 32, F, cols, Z);
    run<128, 2, 54, 21, 21>("t128 v2 21 of 54 from L2", 0, F, cols, Z);
    run<128, 1, 54, 21, 21, 1>("t128 v1 21 of 54 L2 + gate", 0, F, cols, Z);
    run<128, 1, 42, 1>("t128 v1 read only", 0, F, cols, Z);
    run<128, 1, 1, 42>("t128 v1 write only", 0, F, cols, Z);
    return 0;
}

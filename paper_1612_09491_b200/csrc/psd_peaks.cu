// psd_peaks.cu -- roofline-denominator micro-benchmarks (include/psd_peaks.h).  Not on the
// deposit path: these measure what the FP64 pipe, the shared-memory fp64 atomic unit and the L2
// fp64 reduction path of this B200 sustain, so bench.py can quote the deposit kernel against a
// measured peak instead of a datasheet number.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/psd_peaks.h"

namespace {

constexpr int FMA_CHAINS = 8;       // independent accumulators per thread (latency 4-8 cycles)
constexpr int FMA_ITERS = 4096;     // x FMA_CHAINS FMAs per thread
constexpr int FMA_THREADS = 256;

template <class T>
__global__ void __launch_bounds__(FMA_THREADS) k_fma(T* sink, T a, T b) {
    T acc[FMA_CHAINS];
#pragma unroll
    for (int c = 0; c < FMA_CHAINS; ++c) acc[c] = (T)(threadIdx.x + c);
#pragma unroll 1
    for (int it = 0; it < FMA_ITERS / 4; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int c = 0; c < FMA_CHAINS; ++c) acc[c] = acc[c] * a + b;  // contracted to one FMA
    }
    T s = 0;
#pragma unroll
    for (int c = 0; c < FMA_CHAINS; ++c) s += acc[c];
    if (s == (T)-12345.678) sink[0] = s;  // never true for the arguments used; keeps the loop alive
}

constexpr int SA_THREADS = 128;
constexpr int SA_ITERS = 4096;

__global__ void __launch_bounds__(SA_THREADS) k_shared_atomic(double* sink) {
    __shared__ double tile[512];
    for (int i = threadIdx.x; i < 512; i += SA_THREADS) tile[i] = 0.0;
    __syncthreads();
    // lane l of warp w walks the tile with an odd stride: 32 distinct cells per warp instruction,
    // consecutive doubles -> 2-way bank conflict at most (64-bit accesses, 32 banks x 4 B)
    unsigned idx = threadIdx.x * 5u + 1u;
#pragma unroll 4
    for (int it = 0; it < SA_ITERS; ++it) {
        atomicAdd(&tile[idx & 511u], 1.0);
        idx += 37u * 32u + 32u;
    }
    __syncthreads();
    if (tile[threadIdx.x] == -1.0) sink[0] = 1.0;
}

constexpr int GR_THREADS = 128;
constexpr int GR_G = 256;

// pattern 0: flush of an 8^3 tile into a GR_G^3 grid (4 cells per thread)
__global__ void __launch_bounds__(GR_THREADS) k_global_red_tile(double* grid, int rounds) {
    const int nt = GR_G / 8;
    for (int r = 0; r < rounds; ++r) {
        unsigned t = (blockIdx.x * 2654435761u + r * 40503u) % (unsigned)(nt * nt * nt);
        int tz = t % nt, ty = (t / nt) % nt, tx = t / (nt * nt);
        double* base = grid + ((size_t)(tx * 8) * GR_G + ty * 8) * GR_G + tz * 8;
        for (int i = threadIdx.x; i < 512; i += GR_THREADS) {
            int cz = i & 7, cy = (i >> 3) & 7, cx = i >> 6;
            atomicAdd(base + ((size_t)cx * GR_G + cy) * GR_G + cz, 1.0);
        }
    }
}

// pattern 1: one 128-byte line per lane, pseudo-random over `lines` lines
__global__ void __launch_bounds__(GR_THREADS) k_global_red_scatter(double* buf, unsigned long long lines, int rounds) {
    unsigned long long x = (blockIdx.x * (unsigned long long)GR_THREADS + threadIdx.x) * 0x9E3779B97F4A7C15ull + 1ull;
    for (int r = 0; r < rounds; ++r) {
        x ^= x >> 29; x *= 0xBF58476D1CE4E5B9ull; x ^= x >> 32;
        atomicAdd(buf + (x % lines) * 16ull, 1.0);
    }
}

struct Timer {
    cudaEvent_t a = nullptr, b = nullptr;
    cudaStream_t st;
    explicit Timer(cudaStream_t s) : st(s) { cudaEventCreate(&a); cudaEventCreate(&b); }
    ~Timer() { if (a) cudaEventDestroy(a); if (b) cudaEventDestroy(b); }
    template <class F> double best_ms(int reps, F launch) {
        launch();  // warm-up
        double best = 1e300;
        for (int r = 0; r < reps; ++r) {
            cudaEventRecord(a, st);
            launch();
            cudaEventRecord(b, st);
            cudaEventSynchronize(b);
            float ms = 0;
            cudaEventElapsedTime(&ms, a, b);
            if (ms > 0 && ms < best) best = ms;
        }
        return best;
    }
};

int prologue(int device, int reps, double* out, int* sms) {
    if (!out || reps < 1) return 1;
    if (cudaSetDevice(device) != cudaSuccess) return 4;
    if (cudaDeviceGetAttribute(sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) return 4;
    return 0;
}

template <class T>
int run_fma(int device, void* stream, int reps, double* out) {
    int sms = 0;
    if (int rc = prologue(device, reps, out, &sms)) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    T* sink = nullptr;
    if (cudaMalloc(&sink, sizeof(T)) != cudaSuccess) return 4;
    const int grid = sms * 16;
    Timer tm(st);
    double ms = tm.best_ms(reps, [&] { k_fma<T><<<grid, FMA_THREADS, 0, st>>>(sink, (T)1.0000001, (T)1e-9); });
    cudaFree(sink);
    if (cudaGetLastError() != cudaSuccess) return 4;
    *out = 2.0 * (double)grid * FMA_THREADS * FMA_CHAINS * FMA_ITERS / (ms * 1e-3);
    return 0;
}

}  // namespace

extern "C" {

int psd_peak_fp64_fma(int device, void* cuda_stream, int reps, double* out) {
    return run_fma<double>(device, cuda_stream, reps, out);
}

int psd_peak_fp32_fma(int device, void* cuda_stream, int reps, double* out) {
    return run_fma<float>(device, cuda_stream, reps, out);
}

int psd_peak_shared_atomic_f64(int device, void* cuda_stream, int reps, double* out) {
    int sms = 0;
    if (int rc = prologue(device, reps, out, &sms)) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    double* sink = nullptr;
    if (cudaMalloc(&sink, sizeof(double)) != cudaSuccess) return 4;
    const int grid = sms * 16;
    Timer tm(st);
    double ms = tm.best_ms(reps, [&] { k_shared_atomic<<<grid, SA_THREADS, 0, st>>>(sink); });
    cudaFree(sink);
    if (cudaGetLastError() != cudaSuccess) return 4;
    *out = (double)grid * SA_THREADS * SA_ITERS / (ms * 1e-3);
    return 0;
}

int psd_peak_global_red_f64(int device, void* cuda_stream, int pattern, int reps, double* out) {
    int sms = 0;
    if (int rc = prologue(device, reps, out, &sms)) return rc;
    if (pattern != 0 && pattern != 1) return 1;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    double* buf = nullptr;
    const size_t bytes = pattern == 0 ? sizeof(double) * GR_G * GR_G * GR_G : (size_t)1 << 30;
    if (cudaMalloc(&buf, bytes) != cudaSuccess) return 4;
    cudaMemsetAsync(buf, 0, bytes, st);
    Timer tm(st);
    double ms, count;
    if (pattern == 0) {
        const int grid = sms * 32, rounds = 8;
        ms = tm.best_ms(reps, [&] { k_global_red_tile<<<grid, GR_THREADS, 0, st>>>(buf, rounds); });
        count = (double)grid * rounds * 512.0;
    } else {
        const int grid = sms * 32, rounds = 64;
        ms = tm.best_ms(reps, [&] { k_global_red_scatter<<<grid, GR_THREADS, 0, st>>>(buf, bytes / 128, rounds); });
        count = (double)grid * GR_THREADS * rounds;
    }
    cudaFree(buf);
    if (cudaGetLastError() != cudaSuccess) return 4;
    *out = count / (ms * 1e-3);
    return 0;
}

}  // extern "C"

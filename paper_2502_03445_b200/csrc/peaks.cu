// libtqc_peaks.so: micro-benchmarks for the roofline denominators MEASURED_PEAKS.json does not carry (SURVEY.md 8(d):
// "to be measured by the build before any roofline % is quoted"): register-resident FP32 FFMA rate, shared-memory
// LDS.128 bandwidth, L2 read bandwidth.  Not part of the product path; paper_2502_03445_b200/measure_peaks.py drives it
// and writes profiles/peaks_r02.json, which bench.py reads for its `peak` values.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

// 8 independent FMA chains per thread, all in registers
__global__ void __launch_bounds__(1024, 1) ffma_kernel(float *out, int iters, float a, float b) {
    float x0 = threadIdx.x, x1 = x0 + 1.f, x2 = x0 + 2.f, x3 = x0 + 3.f, x4 = x0 + 4.f, x5 = x0 + 5.f, x6 = x0 + 6.f, x7 = x0 + 7.f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
            x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
        }
    }
    const float s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 123.456f) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// every thread reads conflict-free 16-byte words from a 32 KB shared buffer
__global__ void __launch_bounds__(1024, 1) lds_kernel(float *out, int iters) {
    __shared__ __align__(16) float4 buf[2048];
    for (int i = threadIdx.x; i < 2048; i += blockDim.x) buf[i] = make_float4((float)i, 1.f, 2.f, 3.f);
    __syncthreads();
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    int idx = threadIdx.x;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const float4 v = buf[(idx + u * 256) & 2047];
            acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
        }
        idx = (idx + 32) & 2047;
    }
    if (acc.x + acc.y + acc.z + acc.w == 123.456f) out[blockIdx.x * blockDim.x + threadIdx.x] = acc.x;
}

// grid-stride float4 reads of a buffer that fits L2, repeated
__global__ void __launch_bounds__(1024, 2) l2_kernel(const float4 *__restrict__ src, float *out, long long n_vec, int reps) {
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (int r = 0; r < reps; ++r)
        for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_vec; i += stride) {
            const float4 v = __ldcg(src + i);
            acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
        }
    if (acc.x + acc.y + acc.z + acc.w == 123.456f) out[blockIdx.x * blockDim.x + threadIdx.x] = acc.x;
}

// Store-path probe: one 512-thread block per SM writes 128 KB tiles (128 rows x 1024 B of a matrix with `pitch`
// bytes per row, tiles in the pair kernel's order) in one of four warp-store patterns:
//   1  st.v2, a quad of lanes = one 32-byte sector, 8 rows per instruction   (8-byte stores from the tcgen05.ld 16x256b layout)
//   2  st.v4, 8 lanes = one 128-byte line, 4 rows per instruction
//   4  st.v4, a warp writes 512 contiguous bytes of one row
//   5  st.v4, a quad = 64 contiguous bytes of a row, 8 rows per instruction      (16-byte stores after the lane exchange)
template <int PAT>
__global__ void __launch_bounds__(512, 1) store_tiles_kernel(unsigned char *p, long long tiles, size_t pitch) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int w4 = warp & 3, grp = warp >> 2;
    const long long per_row = (long long)(pitch / 1024);
    for (long long t = blockIdx.x; t < tiles; t += gridDim.x) {
        unsigned char *tile = p + (size_t)(t / per_row) * 128 * pitch + (size_t)(t % per_row) * 1024;
        if (PAT == 1) {
#pragma unroll
            for (int h = 0; h < 4; ++h)
#pragma unroll
                for (int g = 0; g < 8; ++g)
                    *reinterpret_cast<float2 *>(tile + (size_t)(32 * w4 + (lane >> 2) + 8 * h) * pitch + 256 * grp + 32 * g + 8 * (lane & 3)) = make_float2(1.f, 2.f);
        } else if (PAT == 2) {
#pragma unroll
            for (int h = 0; h < 8; ++h)
#pragma unroll
                for (int g = 0; g < 2; ++g)
                    *reinterpret_cast<float4 *>(tile + (size_t)(32 * w4 + (lane >> 3) + 4 * h) * pitch + 256 * grp + 128 * g + 16 * (lane & 7)) = make_float4(1.f, 2.f, 3.f, 4.f);
        } else if (PAT == 5) {
#pragma unroll
            for (int h = 0; h < 4; ++h)
#pragma unroll
                for (int g = 0; g < 4; ++g)
                    *reinterpret_cast<float4 *>(tile + (size_t)(32 * w4 + (lane >> 2) + 8 * h) * pitch + 256 * grp + 64 * g + 16 * (lane & 3)) = make_float4(1.f, 2.f, 3.f, 4.f);
        } else {
#pragma unroll
            for (int h = 0; h < 8; ++h)
#pragma unroll
                for (int g = 0; g < 2; ++g)
                    *reinterpret_cast<float4 *>(tile + (size_t)(8 * warp + h) * pitch + 512 * g + 16 * lane) = make_float4(1.f, 2.f, 3.f, 4.f);
        }
    }
}

template <typename F>
int timed(F launch, float *ms) {
    cudaEvent_t a, b;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return -7;
    launch();                                                        // warm-up
    cudaEventRecord(a);
    launch();
    cudaEventRecord(b);
    const cudaError_t e = cudaEventSynchronize(b);
    cudaEventElapsedTime(ms, a, b);
    cudaEventDestroy(a); cudaEventDestroy(b);
    return e == cudaSuccess && cudaGetLastError() == cudaSuccess ? 0 : -7;
}

int sm_count() { int dev = 0, n = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev); return n; }

}  // namespace

extern "C" {

// FP32 FFMA rate in TFLOP/s (2 flops per FMA), one 1024-thread block per SM, `iters` x 128 FMAs per thread
int tqc_peak_ffma(int iters, double *tflops, double *ms_out) {
    float *out = nullptr;
    const int sms = sm_count();
    if (cudaMalloc(&out, (size_t)sms * 1024 * 4) != cudaSuccess) return -7;
    float ms = 0.f;
    const int rc = timed([&] { ffma_kernel<<<sms, 1024>>>(out, iters, 1.0000001f, 1e-9f); }, &ms);
    cudaFree(out);
    if (rc) return rc;
    *tflops = 2.0 * 128.0 * iters * 1024.0 * sms / (ms * 1e-3) / 1e12;
    *ms_out = ms;
    return 0;
}

// shared-memory read bandwidth in GB/s (LDS.128, conflict-free), one 1024-thread block per SM
int tqc_peak_lds(int iters, double *gbs, double *ms_out) {
    float *out = nullptr;
    const int sms = sm_count();
    if (cudaMalloc(&out, (size_t)sms * 1024 * 4) != cudaSuccess) return -7;
    float ms = 0.f;
    const int rc = timed([&] { lds_kernel<<<sms, 1024>>>(out, iters); }, &ms);
    cudaFree(out);
    if (rc) return rc;
    *gbs = 16.0 * 8.0 * iters * 1024.0 * sms / (ms * 1e-3) / 1e9;
    *ms_out = ms;
    return 0;
}

// L2 read bandwidth in GB/s: `bytes` (<= L2 size) read `reps` times by 2 x 1024 threads per SM
int tqc_peak_l2(size_t bytes, int reps, double *gbs, double *ms_out) {
    float4 *src = nullptr;
    float *out = nullptr;
    const int sms = sm_count();
    if (cudaMalloc(&src, bytes) != cudaSuccess || cudaMalloc(&out, (size_t)sms * 2048 * 4) != cudaSuccess) return -7;
    cudaMemset(src, 0, bytes);
    float ms = 0.f;
    const int rc = timed([&] { l2_kernel<<<2 * sms, 1024>>>(src, out, (long long)(bytes / 16), reps); }, &ms);
    cudaFree(src); cudaFree(out);
    if (rc) return rc;
    *gbs = (double)bytes * reps / (ms * 1e-3) / 1e9;
    *ms_out = ms;
    return 0;
}

// store bandwidth in GB/s of `bytes` (a multiple of 128 x pitch) written once in pattern `pattern` (store_tiles_kernel) by
// `blocks` blocks (0: one per SM); pitch = bytes per matrix row, a multiple of 1024
int tqc_peak_store(int pattern, size_t bytes, size_t pitch, int blocks, double *gbs, double *ms_out) {
    if (pitch < 1024 || pitch % 1024 || bytes % (128 * pitch)) return -1;
    unsigned char *buf = nullptr;
    if (cudaMalloc(&buf, bytes) != cudaSuccess) return -7;
    const int nb = blocks > 0 ? blocks : sm_count();
    const long long tiles = (long long)(bytes / (128 * 1024));
    float ms = 0.f;
    int rc = -1;
    if (pattern == 1) rc = timed([&] { store_tiles_kernel<1><<<nb, 512>>>(buf, tiles, pitch); }, &ms);
    else if (pattern == 2) rc = timed([&] { store_tiles_kernel<2><<<nb, 512>>>(buf, tiles, pitch); }, &ms);
    else if (pattern == 4) rc = timed([&] { store_tiles_kernel<4><<<nb, 512>>>(buf, tiles, pitch); }, &ms);
    else if (pattern == 5) rc = timed([&] { store_tiles_kernel<5><<<nb, 512>>>(buf, tiles, pitch); }, &ms);
    cudaFree(buf);
    if (rc) return rc;
    *gbs = (double)bytes / (ms * 1e-3) / 1e9;
    *ms_out = ms;
    return 0;
}

}  // extern "C"

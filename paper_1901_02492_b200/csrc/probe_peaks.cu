// probe_peaks.cu -- microbenchmarks behind the roofline denominators of DESIGN.md section 5.2:
// sample-load rates of the search kernel's inner body (LDS.64 / LDG.64 + add.f32x2 + count) from shared
// memory, L1, L2 and HBM, streaming read bandwidth versus footprint, and TMA box-fill throughput.
// Stand-alone program (not part of libkbmod_b200.so):  nvcc -gencode arch=compute_100a,code=sm_100a -O3 \
//     -o probe_peaks probe_peaks.cu && ./probe_peaks        (see profiles/r01_microbench.md)
// TMA rule learnt the hard way: the box start address must be 16-byte aligned (x coordinate a
// multiple of 4 fp32 elements); an 8-byte aligned start raises "illegal instruction".
#include <cuda_runtime.h>
#include <cuda.h>
#include <cstdio>
#include <cstdlib>
#include <cstdint>
#include <vector>

#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("CUDA error %s at %d\n", cudaGetErrorString(e), __LINE__); exit(1);} } while (0)

__device__ __forceinline__ void acc2(unsigned long long& a, unsigned long long s) {
    asm("add.rn.f32x2 %0, %0, %1;" : "+l"(a) : "l"(s));
}
__device__ __forceinline__ unsigned cnt_add(unsigned c, unsigned long long s) {
    return c + (unsigned)(s >> 63);
}

// MODE 0: LDG (ld.global.nc) ; MODE 1: LDS
// each thread: R rows; per iteration: uniform offset from table; R x (load64, fadd2, count)
template <int R, int MODE>
__global__ void __launch_bounds__(512) gather_kernel(const unsigned long long* __restrict__ buf, size_t span_elems,
                                                     size_t cta_stride_elems, int iters, const int* __restrict__ offs,
                                                     int noffs, int rowpitch, float* out, int smem_elems) {
    extern __shared__ unsigned long long sm[];
    const unsigned long long* base;
    if (MODE == 1) {
        for (int k = threadIdx.x; k < smem_elems; k += blockDim.x) sm[k] = buf[k];
        __syncthreads();
        base = sm + threadIdx.x;
    } else {
        base = buf + ((size_t)blockIdx.x * cta_stride_elems) % span_elems + threadIdx.x;
    }
    unsigned long long a[R];
    unsigned c[R];
#pragma unroll
    for (int r = 0; r < R; ++r) { a[r] = 0ull; c[r] = 0; }
    for (int it = 0; it < iters; ++it) {
        const int o = __ldg(offs + (it % noffs));
        const unsigned long long* p = base + o;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            unsigned long long s;
            if (MODE == 1) s = p[r * rowpitch];
            else s = __ldg(p + (size_t)r * rowpitch);
            acc2(a[r], s);
            c[r] = cnt_add(c[r], s);
        }
    }
    float t = 0;
#pragma unroll
    for (int r = 0; r < R; ++r) t += __uint_as_float((unsigned)a[r]) + __uint_as_float((unsigned)(a[r] >> 32)) + c[r];
    if (t == 123.456f) out[0] = t;
}

// plain streaming read BW (LDG.128), span controls L2 residency
__global__ void __launch_bounds__(512) stream_kernel(const uint4* __restrict__ buf, size_t n, int passes, float* out) {
    unsigned acc = 0;
    for (int p = 0; p < passes; ++p)
        for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (size_t)gridDim.x * blockDim.x) {
            uint4 v = __ldg(buf + k);
            acc += v.x ^ v.y ^ v.z ^ v.w;
        }
    if (acc == 0x12345678u) out[0] = acc;
}

static float timeit(cudaStream_t st, void (*fn)(void*), void* arg, int reps) {
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    fn(arg); fn(arg);
    CK(cudaDeviceSynchronize());
    cudaEventRecord(e0, st);
    for (int r = 0; r < reps; ++r) fn(arg);
    cudaEventRecord(e1, st);
    CK(cudaDeviceSynchronize());
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    return ms / reps;
}

struct GArgs { int R, mode, grid, threads, iters, noffs, rowpitch, smem_elems; size_t span, stride; const unsigned long long* buf; const int* offs; float* out; };
template <int R, int MODE> static void launch_g(const GArgs& g) {
    size_t sh = MODE == 1 ? (size_t)g.smem_elems * 8 : 0;
    cudaFuncSetAttribute(gather_kernel<R, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    gather_kernel<R, MODE><<<g.grid, g.threads, sh>>>(g.buf, g.span, g.stride, g.iters, g.offs, g.noffs, g.rowpitch, g.out, g.smem_elems);
}
static void run_g(void* p) {
    GArgs& g = *(GArgs*)p;
    if (g.mode == 0) { if (g.R == 8) launch_g<8, 0>(g); else launch_g<4, 0>(g); }
    else { if (g.R == 8) launch_g<8, 1>(g); else launch_g<4, 1>(g); }
}
struct SArgs { const uint4* buf; size_t n; int passes; float* out; int grid; };
static void run_s(void* p) { SArgs& s = *(SArgs*)p; stream_kernel<<<s.grid, 512>>>(s.buf, s.n, s.passes, s.out); }
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_3d(unsigned dst, const void* tmap, int c0, int c1, int c2, unsigned bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(dst), "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}

// ---- variant 3: fill throughput; one producer thread per CTA, STAGES-deep ring, random boxes inside a region
template <int STAGES>
__global__ void __launch_bounds__(128) k_fill(const __grid_constant__ CUtensorMap tm, int bytes, int iters, int xr, int yr, int nimg, float* out) {
    extern __shared__ __align__(128) unsigned char smf[];
    __shared__ __align__(8) unsigned long long bar[STAGES];
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) mbar_init(smem_u32(&bar[s]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned rng = blockIdx.x * 2654435761u + 12345u;
        for (int it = 0; it < iters + STAGES; ++it) {
            const int s = it % STAGES;
            if (it >= STAGES) mbar_wait(smem_u32(&bar[s]), ((it / STAGES) - 1) & 1);
            if (it < iters) {
                rng = rng * 1664525u + 1013904223u;
                const int cx = (int)((rng >> 8) % (unsigned)xr) * 4;
                const int cy = (int)((rng >> 20) % (unsigned)yr);
                const int ci = (int)((rng >> 4) % (unsigned)nimg);
                mbar_expect_tx(smem_u32(&bar[s]), bytes);
                tma_3d(smem_u32(smf + (size_t)s * bytes), &tm, cx, cy, ci, smem_u32(&bar[s]));
            }
        }
    }
    __syncthreads();
    if (out && smf[threadIdx.x] == 77 && iters < 0) out[0] = 1;
}

typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                             const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                             CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeFn get_enc() {
    EncodeFn enc = nullptr;
    cudaDriverEntryPointQueryResult qr;
    CK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", (void**)&enc, cudaEnableDefault, &qr));
    if (qr != cudaDriverEntryPointSuccess || !enc) { printf("no cuTensorMapEncodeTiled\n"); exit(1); }
    return enc;
}
static CUtensorMap make_map(EncodeFn enc, void* base, int W, int H, int N, int bw, int bh) {
    CUtensorMap tm;
    cuuint64_t dims[3] = {(cuuint64_t)2 * W, (cuuint64_t)H, (cuuint64_t)N};
    cuuint64_t strides[2] = {(cuuint64_t)2 * W * 4, (cuuint64_t)2 * W * 4 * H};
    cuuint32_t box[3] = {(cuuint32_t)(2 * bw), (cuuint32_t)bh, 1};
    cuuint32_t es[3] = {1, 1, 1};
    CUresult r = enc(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { printf("encode failed %d\n", (int)r); exit(1); }
    return tm;
}

int main() {
    // thr=1024 rows of the original sweep are omitted: the kernels are compiled for <= 512 threads

    const size_t W = 4096, H = 4096, NIMG = 4;
    const size_t nel = W * H * NIMG;               // float2 elements: 512 MB
    unsigned long long* buf; CK(cudaMalloc(&buf, nel * 8));
    CK(cudaMemset(buf, 0, nel * 8));
    float* out; CK(cudaMalloc(&out, 1024));
    int dev_clk; cudaDeviceGetAttribute(&dev_clk, cudaDevAttrClockRate, 0);
    printf("clock attr %d kHz\n", dev_clk);
    const double clk = 1.965e9;

    // ---- stream BW vs span
    for (size_t mb : {16, 32, 64, 96, 128, 256, 512}) {
        SArgs s{(const uint4*)buf, mb * 1024 * 1024 / 16, (int)(2048 / mb) + 1, out, 148 * 4};
        float ms = timeit(0, run_s, &s, 5);
        double bytes = (double)s.n * 16 * s.passes;
        printf("stream span %4zu MB: %.2f TB/s  (%.1f B/clk/SM)\n", mb, bytes / ms / 1e9, bytes / (ms * 1e-3) / clk / 148);
    }
    // ---- gather kernels
    std::vector<int> offs(1024);
    int* doffs; CK(cudaMalloc(&doffs, 4096));
    auto run_gather = [&](const char* name, int R, int mode, int threads, int ctas_per_sm, int iters, int rowpitch,
                          size_t span, size_t stride, int offrange_rows, int offrange_x, int smem_elems) {
        unsigned rng = 1;
        for (auto& o : offs) {
            rng = rng * 1664525u + 1013904223u;
            int oy = offrange_rows ? (rng >> 8) % offrange_rows : 0;
            int ox = offrange_x ? (rng >> 20) % offrange_x : 0;
            o = oy * rowpitch + ox;
        }
        CK(cudaMemcpy(doffs, offs.data(), 4096, cudaMemcpyHostToDevice));
        GArgs g{R, mode, 148 * ctas_per_sm, threads, iters, 1024, rowpitch, smem_elems, span, stride, buf, doffs, out};
        float ms = timeit(0, run_g, &g, 3);
        double samples = (double)g.grid * threads * R * iters;
        printf("%-44s R=%d thr=%d cta/sm=%d: %.3f ms  %.2f samples/clk/SM  (%.1f B/clk/SM, %.2f TB/s)\n", name, R, threads,
               ctas_per_sm, ms, samples / (ms * 1e-3) / clk / 148, samples * 8 / (ms * 1e-3) / clk / 148, samples * 8 / ms / 1e9);
    };
    // LDS: 512 thr, window 544 x (R+40) rows
    for (int thr : {256, 512}) for (int cps : {1, 2}) {
        if (thr * cps > 2048) continue;
        run_gather("LDS.64 smem window", 8, 1, thr, cps, 20000, thr + 32, 0, 0, 8, 32, (thr + 32) * 16);
    }
    run_gather("LDS.64 smem window", 4, 1, 512, 2, 20000, 544, 0, 0, 8, 32, 544 * 16);
    // LDG L1-resident: each CTA hammers a 64 KB region (rowpitch 544)
    for (int cps : {1, 2}) {
        run_gather("LDG.64 L1-hit (64KB/CTA region)", 8, 0, 512, cps, 20000, 544, nel - (1 << 20), 1 << 16, 8, 32, 0);
        run_gather("LDG.64 L1-hit (64KB/CTA region)", 4, 0, 512, cps, 20000, 544, nel - (1 << 20), 1 << 16, 8, 32, 0);
    }
    // LDG L2-resident, L1-miss: rows of image (pitch 4096), offsets over 256 rows x 3000 px: working set per CTA ~ 8 MB; all CTAs share a 32 MB span
    for (int cps : {1, 2, 4}) {
        run_gather("LDG.64 L2-hit (random windows in 32MB)", 8, 0, 512, cps, 4000, 4096, (size_t)4 << 20, 1 << 14, 240, 3000, 0);
    }
    run_gather("LDG.64 L2-hit R=4", 4, 0, 512, 4, 4000, 4096, (size_t)4 << 20, 1 << 14, 240, 3000, 0);
    run_gather("LDG.64 L2-hit thr=256 cps=8", 8, 0, 256, 8, 4000, 4096, (size_t)4 << 20, 1 << 14, 240, 3000, 0);
    // LDG HBM: offsets over entire 512 MB
    run_gather("LDG.64 HBM (random windows in 512MB)", 8, 0, 512, 4, 2000, 4096, nel - ((size_t)40 << 20), 1 << 18, 4000, 3000, 0);

    // ---- TMA box fill (3-D tensor map over [4][4096][4096] float2, zero fill), 4-deep ring, no consumer
    {
        EncodeFn enc = get_enc();
        const int W = 4096, H = 4096, N = 4;
        float* dst = out;
        cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
        CK(cudaFuncSetAttribute(k_fill<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        for (int bh : {32, 48, 64}) for (int bw : {64, 96, 128}) for (int region : {512, 4096}) {
            const int bytes = bw * bh * 8;
            if (bytes * 4 > 200 * 1024) continue;
            CUtensorMap tm = make_map(enc, buf, W, H, N, bw, bh);
            const int iters = 4000;
            for (int rep = 0; rep < 2; ++rep) {
                cudaEventRecord(e0);
                k_fill<4><<<148, 128, bytes * 4>>>(tm, bytes, iters, (region - bw) / 2, region - bh, N, dst);
                cudaEventRecord(e1);
                CK(cudaDeviceSynchronize());
            }
            float ms; cudaEventElapsedTime(&ms, e0, e1);
            const double b = (double)148 * iters * bytes;
            printf("TMA fill box %3dx%2d (%2d KB) region %4d^2 x%d img (%4.0f MB): %.3f ms  %.2f TB/s (%.1f B/clk/SM @1.965GHz)\n", bw, bh,
                   bytes / 1024, region, N, (double)region * region * 8 * N / 1e6, ms, b / ms / 1e9, b / (ms * 1e-3) / 1.965e9 / 148);
        }
    }
    CK(cudaDeviceSynchronize());
    printf("done\n");
    return 0;
}

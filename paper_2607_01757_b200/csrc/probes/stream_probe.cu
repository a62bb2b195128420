// stream_probe.cu — read-bandwidth probes behind DESIGN.md 7.1: how fast can one B200 stream the c5 score
// maps (64 x 1080 x 1920 f32 = 531 MB) with (a) plain 16-byte loads, (b) 1-D bulk copies, (c) 3-D tensor-map
// boxes of several shapes, each warp running its own 2-deep mbarrier ring (the structure of k_nms_tma)?
// Not part of libdkd.  Build + run (one GPU):
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 --extended-lambda \
//        -o /tmp/stream_probe paper_2607_01757_b200/csrc/probes/stream_probe.cu -lcuda && /tmp/stream_probe
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdio.h>
#include <stdint.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("err %s line %d\n",cudaGetErrorString(e),__LINE__);return 1;}}while(0)
typedef CUresult (*PFN)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
__device__ __forceinline__ uint32_t su32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__global__ void k_ldg(const float4* __restrict__ p, size_t n, float* out) {
    float s = 0;
    size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x, st = (size_t)gridDim.x * blockDim.x;
    for (; i + 3 * st < n; i += 4 * st) {
        float4 a = __ldcs(p + i), b = __ldcs(p + i + st), c = __ldcs(p + i + 2 * st), d = __ldcs(p + i + 3 * st);
        s += a.x + b.y + c.z + d.w;
    }
    for (; i < n; i += st) s += __ldcs(p + i).x;
    if (s == 123.456f) out[0] = s;
}
// 1-D bulk copies: each warp streams CH-byte chunks through a 2-stage ring
template <int CH>
__global__ void k_bulk(const unsigned char* __restrict__ p, size_t nchunks, float* out, int warps) {
    extern __shared__ __align__(128) unsigned char sm[];
    __shared__ __align__(8) uint64_t bars[64];
    int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned char* my = sm + warp * 2 * CH;
    uint64_t* bar = bars + warp * 2;
    size_t first = blockIdx.x * (size_t)warps + warp, step = (size_t)gridDim.x * warps;
    long n_my = first < nchunks ? (long)((nchunks - first + step - 1) / step) : 0;
    if (lane == 0) {
        for (int s = 0; s < 2; ++s) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(su32(&bar[s])));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
    auto issue = [&](long it) {
        if (lane == 0) {
            int s = it & 1;
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(su32(&bar[s])), "r"(CH) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(su32(my + s * CH)), "l"(p + (first + it * step) * CH), "r"(CH), "r"(su32(&bar[s])) : "memory");
        }
    };
    for (long it = 0; it < 2 && it < n_my; ++it) issue(it);
    float acc = 0;
    for (long it = 0; it < n_my; ++it) {
        int s = it & 1; uint32_t par = (it >> 1) & 1;
        asm volatile("{\n.reg .pred P1;\nW:\nmbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n@P1 bra D;\nbra W;\nD:\n}" ::"r"(su32(&bar[s])), "r"(par) : "memory");
        acc += reinterpret_cast<float*>(my + s * CH)[lane];
        __syncwarp();
        if (it + 2 < n_my) issue(it + 2);
    }
    if (acc == 123.456f) out[0] = acc;
}
// each warp streams boxes (bw x bh) in raster order through a 2-stage ring; sw = strip step in x, sh = step in y
__global__ void k_box(const __grid_constant__ CUtensorMap tm, int box_bytes, int sx, int sy, int nx, int ny, int nb, float* out, int warps) {
    extern __shared__ __align__(128) unsigned char sm[];
    __shared__ __align__(8) uint64_t bars[64];
    int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned char* my = sm + (size_t)warp * 2 * box_bytes;
    uint64_t* bar = bars + warp * 2;
    long total = (long)nx * ny * nb;
    long first = blockIdx.x * (long)warps + warp, step = (long)gridDim.x * warps;
    long n_my = first < total ? (total - first + step - 1) / step : 0;
    if (lane == 0) {
        for (int s = 0; s < 2; ++s) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(su32(&bar[s])));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
    auto issue = [&](long it) {
        if (lane == 0) {
            long t = first + it * step;
            int b = t / ((long)nx * ny); int rem = t - (long)b * nx * ny; int ty = rem / nx, tx = rem - ty * nx;
            int s = it & 1;
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(su32(&bar[s])), "r"(box_bytes) : "memory");
            asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                ::"r"(su32(my + s * box_bytes)), "l"((uint64_t)&tm), "r"(su32(&bar[s])), "r"(tx * sx - 4), "r"(ty * sy), "r"(b) : "memory");
        }
    };
    for (long it = 0; it < 2 && it < n_my; ++it) issue(it);
    float acc = 0;
    for (long it = 0; it < n_my; ++it) {
        int s = it & 1; uint32_t par = (it >> 1) & 1;
        asm volatile("{\n.reg .pred P1;\nW:\nmbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n@P1 bra D;\nbra W;\nD:\n}" ::"r"(su32(&bar[s])), "r"(par) : "memory");
        acc += reinterpret_cast<float*>(my + s * box_bytes)[lane];
        __syncwarp();
        if (it + 2 < n_my) issue(it + 2);
    }
    if (acc == 123.456f) out[0] = acc;
}
__global__ void k_fill(uint32_t* p, size_t n) { size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; size_t st = (size_t)gridDim.x * blockDim.x; for (; i < n; i += st) { uint32_t h = (uint32_t)i * 2654435761u; h ^= h >> 15; h *= 2246822519u; h ^= h >> 13; p[i] = 0x3d000000u + (h & 0x7fffffu); } }
int main(int argc, char** argv) {
    (void)argv;
    const int B = 64, H = 1080, W = 1920;
    size_t bytes = (size_t)B * H * W * 4;
    unsigned char* d; float* o;
    CK(cudaMalloc(&d, bytes)); CK(cudaMalloc(&o, 4)); CK(cudaMemset(d, 1, bytes)); if (argc > 1) { k_fill<<<148*8, 512>>>((uint32_t*)d, bytes / 4); CK(cudaDeviceSynchronize()); printf("random fill\n"); }
    void* fn; cudaDriverEntryPointQueryResult q;
    CK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q));
    PFN enc = (PFN)fn;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    CK(cudaFuncSetAttribute(k_box, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024));
    auto run = [&](int bw, int bh, int sx, int warps, int ctas, CUtensorMapL2promotion prom, const char* pn) {
        CUtensorMap tm;
        cuuint64_t dims[3] = {(cuuint64_t)W, (cuuint64_t)H, (cuuint64_t)B};
        cuuint64_t strides[2] = {(cuuint64_t)W * 4, (cuuint64_t)W * H * 4};
        cuuint32_t box[3] = {(cuuint32_t)bw, (cuuint32_t)bh, 1}; cuuint32_t es[3] = {1, 1, 1};
        CUresult r = enc(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, d, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, prom, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) { printf("encode fail %d\n", (int)r); return; }
        int nx = (W + sx - 1) / sx, ny = (H + bh - 1) / bh, bb = bw * bh * 4;
        int smem = warps * 2 * bb;
        auto f = [&] { k_box<<<148 * ctas, warps * 32, smem>>>(tm, bb, sx, bh, nx, ny, B, o, warps); };
        for (int i = 0; i < 3; ++i) f();
        cudaEventRecord(e0); for (int i = 0; i < 20; ++i) f(); cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1); ms /= 20;
        float ms1 = 0; for (int i = 0; i < 10; ++i) { cudaEventRecord(e0); f(); cudaEventRecord(e1); cudaEventSynchronize(e1); float m; cudaEventElapsedTime(&m, e0, e1); ms1 += m / 10; }
        printf("single-launch %7.1f us | ", ms1 * 1e3);
        printf("box %3dx%-2d step %3d  %2d warps x %d CTA/SM  %s: %7.1f us  %7.1f GB/s algorithmic (%s)\n", bw, bh, sx, warps, ctas, pn, ms * 1e3, bytes / ms / 1e6, cudaGetErrorString(cudaGetLastError()));
    };
    {
        auto timeit = [&](const char* name, auto f) {
            for (int i = 0; i < 3; ++i) f();
            cudaEventRecord(e0); for (int i = 0; i < 20; ++i) f(); cudaEventRecord(e1); cudaEventSynchronize(e1);
            float ms; cudaEventElapsedTime(&ms, e0, e1); ms /= 20;
            printf("%-34s %8.1f us  %7.1f GB/s  (%s)\n", name, ms * 1e3, bytes / ms / 1e6, cudaGetErrorString(cudaGetLastError()));
        };
        timeit("linear ld.global.v4, 4 CTA/SM x 512", [&] { k_ldg<<<148 * 4, 512>>>((const float4*)d, bytes / 16, o); });
        auto bulk = [&](auto kern, int CH, int warps, int ctas, const char* nm) {
            cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, warps * 2 * CH);
            timeit(nm, [&] { kern<<<148 * ctas, warps * 32, warps * 2 * CH>>>(d, bytes / CH, o, warps); });
        };
        bulk(k_bulk<8192>, 8192, 6, 2, "1-D bulk 8 KB, 12 warps/SM");
        bulk(k_bulk<4096>, 4096, 10, 2, "1-D bulk 4 KB, 20 warps/SM");
        bulk(k_bulk<2048>, 2048, 16, 2, "1-D bulk 2 KB, 32 warps/SM");
    }
    auto P128 = CU_TENSOR_MAP_L2_PROMOTION_L2_128B; auto P256 = CU_TENSOR_MAP_L2_PROMOTION_L2_256B;
    run(128, 8, 120, 10, 2, P128, "L2_128B");

    run(128, 16, 120, 6, 2, P128, "L2_128B");
    run(128, 16, 120, 6, 2, P256, "L2_256B");
    run(128, 32, 120, 3, 2, P256, "L2_256B");
    run(256, 8, 240, 6, 2, P128, "L2_128B");
    run(256, 8, 240, 6, 2, P256, "L2_256B");
    run(256, 8, 256, 6, 2, P256, "L2_256B");
    run(256, 16, 240, 3, 2, P256, "L2_256B");
    run(248, 8, 240, 6, 2, P256, "L2_256B");
    run(256, 4, 240, 12, 2, P256, "L2_256B");
    run(64, 16, 56, 12, 2, P128, "L2_128B");
    return 0;
}

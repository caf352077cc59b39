// read-bandwidth probe: how fast can 148 persistent CTAs pull random 73,728-B pages into shared memory?
// modes: 0 = 3-D TMA box (64,64,9) per page, 1 = 1-D bulk copy of the contiguous page, 2 = 9 boxes (64,64,1)
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdint>
#include <cstdlib>
#include <vector>
#include <algorithm>
#include <random>
#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("%s: %s\n", #x, cudaGetErrorString(e)); exit(1); } } while (0)
constexpr int kPageBytes = 73728;
__device__ __forceinline__ uint32_t s32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, int n) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(s32(b)), "r"(n)); }
__device__ __forceinline__ void expect(uint64_t* b, uint32_t n) { asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(s32(b)), "r"(n) : "memory"); }
__device__ __forceinline__ void wait(uint64_t* b, uint32_t ph) {
    asm volatile("{\n.reg .pred p;\nW: mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@!p bra W;\n}" ::"r"(s32(b)), "r"(ph) : "memory");
}
template <int MODE, int STAGES>
__global__ void __launch_bounds__(128, 1) rd(const __grid_constant__ CUtensorMap m9, const __grid_constant__ CUtensorMap m1, const uint8_t* pool,
                                             const int* pages, int per_cta, int hold) {
    extern __shared__ uint8_t raw[];
    uint8_t* base = (uint8_t*)(((uintptr_t)raw + 1023) & ~uintptr_t(1023));
    __shared__ uint64_t full[STAGES];
    if (threadIdx.x == 0) {
        for (int i = 0; i < STAGES; ++i) mbar_init(&full[i], 1);
        asm volatile("fence.mbarrier_init.release.cluster;");
    }
    __syncthreads();
    if (threadIdx.x != 0) return;
    const int* pp = pages + blockIdx.x * per_cta;
    auto issue = [&](int i) {
        const int st = i % STAGES;
        const int pid = pp[i];
        expect(&full[st], kPageBytes);
        uint8_t* dst = base + st * kPageBytes;
        if (MODE == 0) {
            asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(s32(dst)),
                         "l"((uint64_t)&m9), "r"(s32(&full[st])), "r"(0), "r"(pid * 64), "r"(0) : "memory");
        } else if (MODE == 1) {
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(s32(dst)),
                         "l"(pool + size_t(pid) * kPageBytes), "r"(kPageBytes), "r"(s32(&full[st])) : "memory");
        } else {
            for (int c = 0; c < 9; ++c)
                asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
                                 s32(dst + c * 8192)),
                             "l"((uint64_t)&m1), "r"(s32(&full[st])), "r"(0), "r"(pid * 64), "r"(c) : "memory");
        }
    };
    for (int i = 0; i < STAGES && i < per_cta; ++i) issue(i);
    for (int i = 0; i < per_cta; ++i) {
        wait(&full[i % STAGES], (i / STAGES) & 1);
        if (hold) { const long long t = clock64(); while (clock64() - t < hold) {} }
        if (i + STAGES < per_cta) issue(i + STAGES);
    }
}
typedef CUresult (*Enc)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                        CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
template <int MODE, int STAGES>
void run(const CUtensorMap& m9, const CUtensorMap& m1, uint8_t* pool, int* dpages, int per_cta, int grid, const char* name, int hold = 0) {
    const int smem = STAGES * kPageBytes + 1024;
    CK(cudaFuncSetAttribute(rd<MODE, STAGES>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    cudaEvent_t a, b;
    cudaEventCreate(&a); cudaEventCreate(&b);
    float best = 1e9;
    for (int r = 0; r < 6; ++r) {
        cudaEventRecord(a);
        rd<MODE, STAGES><<<grid, 128, smem>>>(m9, m1, pool, dpages + (r % 3) * grid * per_cta, per_cta, hold);
        cudaEventRecord(b);
        CK(cudaEventSynchronize(b));
        float ms; cudaEventElapsedTime(&ms, a, b);
        if (r > 0) best = std::min(best, ms);
    }
    const double bytes = double(grid) * per_cta * kPageBytes;
    printf("%-28s hold %d stages %d grid %d: %.1f us  %.2f TB/s\n", name, hold, STAGES, grid, best * 1e3, bytes / best / 1e9);
}
int main() {
    const int grid = 148, per_cta = 56, sets = 3;
    const int n_pages = grid * per_cta * sets;  // 24,864 pages = 1.83 GB
    uint8_t* pool; CK(cudaMalloc(&pool, size_t(n_pages) * kPageBytes));
    CK(cudaMemset(pool, 1, size_t(n_pages) * kPageBytes));
    std::vector<int> pages(n_pages);
    for (int i = 0; i < n_pages; ++i) pages[i] = i;
    std::mt19937 rng(1);
    std::vector<int> seq = pages;
    std::shuffle(pages.begin(), pages.end(), rng);
    int *dpages, *dseq;
    CK(cudaMalloc(&dpages, n_pages * 4)); CK(cudaMemcpy(dpages, pages.data(), n_pages * 4, cudaMemcpyHostToDevice));
    CK(cudaMalloc(&dseq, n_pages * 4)); CK(cudaMemcpy(dseq, seq.data(), n_pages * 4, cudaMemcpyHostToDevice));
    void* fn; cudaDriverEntryPointQueryResult q;
    CK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q));
    Enc enc = (Enc)fn;
    CUtensorMap m9, m1;
    cuuint64_t dims[3] = {64, cuuint64_t(n_pages) * 64, 9};
    cuuint64_t strides[2] = {1152, 128};
    cuuint32_t es[3] = {1, 1, 1};
    cuuint32_t b9[3] = {64, 64, 9}, b1[3] = {64, 64, 1};
    if (enc(&m9, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, pool, dims, strides, b9, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE)) { printf("enc9 failed\n"); return 1; }
    if (enc(&m1, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, pool, dims, strides, b1, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE)) { printf("enc1 failed\n"); return 1; }
    run<0, 2>(m9, m1, pool, dpages, per_cta, grid, "tma 3d box9 random");
    run<0, 3>(m9, m1, pool, dpages, per_cta, grid, "tma 3d box9 random");
    run<1, 2>(m9, m1, pool, dpages, per_cta, grid, "bulk 1d random");
    run<1, 3>(m9, m1, pool, dpages, per_cta, grid, "bulk 1d random");
    run<2, 3>(m9, m1, pool, dpages, per_cta, grid, "tma 9 x box1 random");
    run<0, 1>(m9, m1, pool, dpages, per_cta, grid, "tma 3d box9 random");
    run<0, 1>(m9, m1, pool, dpages, per_cta, 16, "tma 3d box9 random");
    run<0, 2>(m9, m1, pool, dpages, per_cta, 16, "tma 3d box9 random");
    for (int h = 1000; h <= 4000; h += 1000) {
        run<0, 2>(m9, m1, pool, dpages, per_cta, grid, "tma 3d box9 random", h);
        run<0, 3>(m9, m1, pool, dpages, per_cta, grid, "tma 3d box9 random", h);
    }
    run<0, 3>(m9, m1, pool, dseq, per_cta, grid, "tma 3d box9 sequential");
    run<1, 3>(m9, m1, pool, dseq, per_cta, grid, "bulk 1d sequential");
    return 0;
}

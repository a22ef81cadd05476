// afs_static.cu -- afs_round_count_static: the rounding / satisfied-count step (S9) for callers that are not
// allowed to allocate device memory when they make the call.
//
// Who that is: code running where a cudaMalloc is either forbidden or too costly -- a solver loop embedded in a host
// program whose framework has already handed all of HBM to its own pool allocator (a cudaMalloc then fails, or forces
// the pool to give memory back), a latency-bound service thread (cudaMalloc / cudaFree synchronise the whole device
// and stall every other stream), or a plug-in whose contract with its host says "no driver allocations after set-up".
// The ordinary afs_round_count keeps its transposed working copy of X in the handle's workspace, which it (re)allocates
// with cudaMalloc the first time a larger batch is seen; that first call is the one such callers cannot make.
//
// Here the working memory is ONE file-scope device array of fixed size, part of the library image: every GPU that loads
// libafs_b200.so holds AFS_STATIC_SCRATCH_BYTES of it until the process exits, used or not.  The entry point calls no
// cudaMalloc, cudaFree or allocating library routine (cudaMemsetAsync / cudaMemcpyAsync on existing memory and kernel
// launches only), and nothing in the handle's workspace is touched or grown.
#include <mutex>

#include "afs_kernels.cuh"
#include "afs_launch.h"

using namespace afs;

// The scratch itself.  In HOST code the name `g_static_scratch` is only a stand-in the runtime uses to look the symbol
// up; it is not a device address and must never be handed to a kernel.  Host code gets the real address once per device
// from cudaGetSymbolAddress (static_scratch_ptr below).
static __device__ __align__(256) unsigned char g_static_scratch[AFS_STATIC_SCRATCH_BYTES];

namespace {

constexpr int MAX_DEVICES = 64;
std::mutex g_ptr_mutex;
unsigned char* g_ptr[MAX_DEVICES] = {nullptr};   // device address of g_static_scratch on each device, once looked up

// Set-up, once per device, with that device current (the caller has made it so).  A module's globals have one
// instance per device, so the address is looked up per device and never reused across devices.
afs_status static_scratch_ptr(int device, unsigned char** out)
{
    if (device < 0 || device >= MAX_DEVICES) return AFS_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_ptr_mutex);
    if (!g_ptr[device]) {
        void* ptr = nullptr;
        CU(cudaGetSymbolAddress(&ptr, g_static_scratch));
        g_ptr[device] = (unsigned char*)ptr;
    }
    *out = g_ptr[device];
    return AFS_OK;
}

size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

// k_count with both of its working arrays in the static scratch: the transposed iterate XT[n][Bp] it reads and the
// per-column counter row it accumulates into (integer atomics, so the sums do not depend on the order).  Thread =
// (constraint, restart), lanes over restarts, as in k_count; there is no retirement state on this path.
__global__ void __launch_bounds__(256) k_count_static(const CountCon* __restrict__ cons, const uint32_t* __restrict__ lits,
                                                      int m, const unsigned char* __restrict__ scratch, size_t xt_off,
                                                      int Bp, int32_t* __restrict__ cnt_row)
{
    __shared__ int s_sat[8][32];
    const float* __restrict__ XT = (const float*)(scratch + xt_off);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int b = blockIdx.y * 32 + lane;
    int cnt = 0;
    for (int c = blockIdx.x * 8 + warp; c < m; c += gridDim.x * 8) {
        CountCon cc = cons[c];
        int t = 0;
        for (int j = 0; j < cc.L; ++j) {
            uint32_t w = lits[cc.off + j];
            float x = ldx(XT, w, Bp, b);
            t += ((x < 0.0f) != ((w >> 31) != 0)) ? 1 : 0;
        }
        cnt += pred(cc.type, cc.L, cc.k, t) ? 1 : 0;
    }
    s_sat[warp][lane] = cnt;
    __syncthreads();
    if (warp == 0) {
        int tot = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) tot += s_sat[w][lane];
        if (tot) atomicAdd(&cnt_row[b], tot);
    }
}

}  // namespace

extern "C" afs_status afs_round_count_static(afs_problem* P, const float* X, int32_t B, int8_t* assign, int32_t* sat,
                                             void* stream)
{
    if (!P || B < 1 || !X || !sat) return AFS_ERR_INVALID_ARG;
    const int Bp = ((B + 31) / 32) * 32;
    // scratch layout: [0, cnt_bytes) the counter row int32[Bp]; [xt_off, xt_off + n Bp 4) the transposed iterate
    const size_t cnt_bytes = (size_t)Bp * sizeof(int32_t);
    const size_t xt_off = align256(cnt_bytes);
    const unsigned long long need = (unsigned long long)xt_off + (unsigned long long)P->n * (unsigned long long)Bp * sizeof(float);
    if (need > (unsigned long long)AFS_STATIC_SCRATCH_BYTES) return AFS_ERR_STATIC_LIMIT;

    DeviceScope dev_scope(P);
    if (cudaSetDevice(P->device) != cudaSuccess) { (void)cudaGetLastError(); return AFS_ERR_CUDA; }
    unsigned char* scratch = nullptr;
    afs_status s = static_scratch_ptr(P->device, &scratch);   // the first call on a device does the look-up
    if (s != AFS_OK) return s;

    cudaStream_t st = (cudaStream_t)stream;
    int32_t* cnt_row = (int32_t*)scratch;
    float* XT = (float*)(scratch + xt_off);
    const int tiles = Bp / 32;
    // the array keeps whatever the previous call left: the counters must start at zero; XT is fully rewritten
    CU(cudaMemsetAsync(cnt_row, 0, cnt_bytes, st));
    dim3 tg((P->n + 31) / 32, tiles);
    k_transpose_in<float><<<tg, 256, 0, st>>>(X, XT, B, P->n, Bp, nullptr, nullptr, nullptr);
    if (P->m > 0) {
        int gx = (P->m + 7) / 8;
        int cap = (P->sm_count * 8 + tiles - 1) / tiles;
        if (gx > cap) gx = cap < 1 ? 1 : cap;
        k_count_static<<<dim3(gx, tiles), 256, 0, st>>>(P->d_count, P->d_count_lits, P->m, scratch, xt_off, Bp, cnt_row);
    }
    CU(cudaMemcpyAsync(sat, cnt_row, (size_t)B * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
    if (assign) k_assign_out<float><<<tg, 256, 0, st>>>(XT, assign, B, P->n, Bp);
    CU(cudaGetLastError());
    return AFS_OK;
}

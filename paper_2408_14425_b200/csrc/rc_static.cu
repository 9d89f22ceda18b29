// rc_static.cu — rc_count_empty_cells_static: the one entry point of librc.so that needs no memory from anybody.
//
// Everything else in the library works out of a workspace the caller lends (rc_set_workspace).  That is no help to a
// caller who has no device memory left to lend and cannot get more: a plug-in inside a host application whose allocator
// took the whole GPU at start-up (cudaMalloc then simply fails), a step inside somebody else's real-time or serving loop
// where cudaMalloc / cudaFree are banned because they synchronise the whole device, or a tool that is only handed the two
// input arrays.  For those callers this file keeps the scratch memory of ONE operation - the empty-cell count that
// rc_analyse_atmosphere bases its "is this atmosphere sparse?" decision on (free-space acceleration) - in a
// fixed array inside the library image itself.  The price: the array (RC_STATIC_MAX_CELLS ints + 256 bytes, about 4 MiB)
// is resident on every GPU that loads the library until the process exits, the problem size is capped, and all calls
// share it.
//
// Nothing in this file is used by, or uses, the context-based path (rc_api.cu / rc_kernels.cu).
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "../../include/rc.h"

namespace {

constexpr int HEADER_BYTES = 256;  // [0, 8): occupied-cell counter, [8, 12): block ticket; the marks start at byte 256
constexpr int MAX_DEVICES = 64;
constexpr int BLOCK = 256;

// The scratch itself.  One copy per GPU that loads this module; lives until the process ends.  Shared by every call.
// NOTE for whoever edits the host code below: in HOST code the name `rc_static_scratch` is only a handle for the
// runtime (a host-side shadow symbol), NOT a device address.  Handing it to a kernel or to cudaMemsetAsync makes them
// fault - or, on systems where the GPU can reach host memory, quietly work on the wrong bytes.  The device address comes
// from cudaGetSymbolAddress, asked once per device with that device current (scratch_address below).
static __device__ __align__(256) unsigned char rc_static_scratch[HEADER_BYTES + sizeof(int) * (size_t)RC_STATIC_MAX_CELLS];

std::mutex g_setup_lock;
void *g_scratch_addr[MAX_DEVICES];  // device address of rc_static_scratch on device d; null = not asked yet
bool g_is_sm100[MAX_DEVICES];

int report(char *errbuf, size_t errbuf_len, int code, const char *fmt, ...) {
    if (errbuf != nullptr && errbuf_len > 0) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(errbuf, errbuf_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// One-time set-up per device; `device` must be current.  No allocation: the array came with the module.
int scratch_address(int device, unsigned char **out, char *errbuf, size_t errbuf_len) {
    std::lock_guard<std::mutex> hold(g_setup_lock);
    if (g_scratch_addr[device] == nullptr) {
        int major = 0;
        cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device);
        if (e != cudaSuccess) {
            cudaGetLastError();
            return report(errbuf, errbuf_len, RC_ERR_CUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
        }
        g_is_sm100[device] = major == 10;
        if (!g_is_sm100[device])
            return report(errbuf, errbuf_len, RC_ERR_NO_DEVICE, "device %d is compute capability %d.x; librc.so holds sm_100a code only", device, major);
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, rc_static_scratch);
        if (e != cudaSuccess || p == nullptr) {
            cudaGetLastError();
            return report(errbuf, errbuf_len, RC_ERR_CUDA, "cudaGetSymbolAddress(rc_static_scratch) on device %d: %s", device, cudaGetErrorString(e));
        }
        g_scratch_addr[device] = p;
    }
    *out = static_cast<unsigned char *>(g_scratch_addr[device]);
    return RC_OK;
}

// A variant of the occupancy scan of rc_analyse_atmosphere (mark_occupied_kernel + occupancy_kernel in rc_kernels.cu)
// folded into one launch.  The arrays are read once, coalesced, W floats per thread (a "chunk"); a thread that finds a
// non-zero value in a cell of interest claims that cell's mark (scratch, zero at launch) and the claimant counts it.  The
// last block to finish turns the count into the answer, so no second launch and no host round trip are needed.
//   chunks [0, nchunk) belong to chi, [nchunk, 2 nchunk) to eta; cell = chunk / chunks_per_cell
template <int W>
__global__ void __launch_bounds__(BLOCK) count_empty_static_kernel(const float *__restrict__ chi, const float *__restrict__ eta,
                                                                   const unsigned char *__restrict__ active, long long nchunk,
                                                                   int chunks_per_cell, long long ncell, unsigned char *scratch,
                                                                   unsigned long long *nempty_out) {
    unsigned long long *noccupied = reinterpret_cast<unsigned long long *>(scratch);
    unsigned *ticket = reinterpret_cast<unsigned *>(scratch + 8);
    int *mark = reinterpret_cast<int *>(scratch + HEADER_BYTES);
    unsigned mine = 0;
    for (long long i = (long long)blockIdx.x * BLOCK + threadIdx.x; i < 2 * nchunk; i += (long long)gridDim.x * BLOCK) {
        const bool second = i >= nchunk;
        const long long j = second ? i - nchunk : i;
        const float *f = second ? eta : chi;
        bool nz;
        if constexpr (W == 4) {
            const float4 v = __ldg(reinterpret_cast<const float4 *>(f) + j);
            nz = v.x != 0.f || v.y != 0.f || v.z != 0.f || v.w != 0.f;
        } else {
            nz = __ldg(f + j) != 0.f;
        }
        if (!nz) continue;
        const long long cell = j / chunks_per_cell;
        if (active != nullptr && __ldg(active + cell) == 0) continue;  // not a cell of interest: empty by definition
        // the plain read only spares the atomic unit: whoever swaps 0 -> 1 is the one thread that counts the cell
        if (*reinterpret_cast<volatile int *>(mark + cell) == 0 && atomicExch(mark + cell, 1) == 0) mine++;
    }
    for (int o = 16; o > 0; o >>= 1) mine += __shfl_down_sync(0xffffffffu, mine, o);
    if ((threadIdx.x & 31) == 0 && mine != 0) atomicAdd(noccupied, (unsigned long long)mine);
    // last block out writes the result
    __shared__ bool last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (last && threadIdx.x == 0) {
        __threadfence();
        *nempty_out = (unsigned long long)ncell - atomicAdd(noccupied, 0ull);
    }
}

}  // namespace

extern "C" int rc_count_empty_cells_static(int device, const float *chi, const float *eta, const unsigned char *active, int nx, int ny,
                                           int nlambda, unsigned long long *nempty_out, void *cuda_stream, char *errbuf,
                                           size_t errbuf_len) {
    if (errbuf != nullptr && errbuf_len > 0) errbuf[0] = '\0';
    if (chi == nullptr || eta == nullptr || nempty_out == nullptr)
        return report(errbuf, errbuf_len, RC_ERR_NULL_ARG, "rc_count_empty_cells_static: chi, eta and nempty_out must not be null");
    if (nx < 1 || ny < 1 || nlambda < 1 || nx > RC_MAX_DIM || ny > RC_MAX_DIM)
        return report(errbuf, errbuf_len, RC_ERR_BAD_SHAPE, "rc_count_empty_cells_static: bad shape %d x %d x %d", nx, ny, nlambda);
    const long long ncell = (long long)nx * ny;
    if (ncell > (long long)RC_STATIC_MAX_CELLS)
        return report(errbuf, errbuf_len, RC_ERR_BAD_SHAPE,
                      "rc_count_empty_cells_static: %d x %d = %lld cells exceed RC_STATIC_MAX_CELLS = %d, the size of the scratch array "
                      "built into librc.so; use rc_analyse_atmosphere with a lent workspace for larger grids",
                      nx, ny, ncell, (int)RC_STATIC_MAX_CELLS);
    if (device < 0 || device >= MAX_DEVICES)
        return report(errbuf, errbuf_len, RC_ERR_NO_DEVICE, "rc_count_empty_cells_static: device %d out of range", device);
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return report(errbuf, errbuf_len, RC_ERR_NO_DEVICE, "cudaSetDevice(%d): %s", device, cudaGetErrorString(e));
    }
    unsigned char *scratch = nullptr;
    const int rc = scratch_address(device, &scratch, errbuf, errbuf_len);
    if (rc != RC_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);

    // The array still holds the previous call's marks and counters: counter, ticket and the marks of this grid start at 0.
    e = cudaMemsetAsync(scratch, 0, HEADER_BYTES + sizeof(int) * (size_t)ncell, st);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return report(errbuf, errbuf_len, RC_ERR_CUDA, "cudaMemsetAsync(scratch): %s", cudaGetErrorString(e));
    }
    const bool vec4 = nlambda % 4 == 0 && ((reinterpret_cast<uintptr_t>(chi) | reinterpret_cast<uintptr_t>(eta)) & 15) == 0;
    const int chunks_per_cell = vec4 ? nlambda / 4 : nlambda;
    const long long nchunk = ncell * chunks_per_cell;
    const long long want = (2 * nchunk + BLOCK - 1) / BLOCK;
    const unsigned blocks = (unsigned)(want < 148LL * 16 ? want : 148LL * 16);  // grid-stride beyond 16 blocks per SM
    if (vec4)
        count_empty_static_kernel<4><<<blocks, BLOCK, 0, st>>>(chi, eta, active, nchunk, chunks_per_cell, ncell, scratch, nempty_out);
    else
        count_empty_static_kernel<1><<<blocks, BLOCK, 0, st>>>(chi, eta, active, nchunk, chunks_per_cell, ncell, scratch, nempty_out);
    e = cudaGetLastError();
    if (e != cudaSuccess) return report(errbuf, errbuf_len, RC_ERR_CUDA, "count_empty_static_kernel launch: %s", cudaGetErrorString(e));
    return RC_OK;
}

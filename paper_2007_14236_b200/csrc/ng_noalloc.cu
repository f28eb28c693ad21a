// =====================================================================================
// ng_noalloc.cu — ng_deliver_noalloc: one step of spike delivery (a3) that allocates nothing.
//
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that
// forbid it).  A variant of delivery kernel 1 (one warp walks a spiking row chunk by chunk) whose scratch —
// the per-target delay ring of ring_slots planes — lives in a file-scope static __device__ array instead
// of memory from ng_allocator / cudaMalloc.  Every GPU that loads libng.so holds the array (16 MiB) until exit.
//
// The array's NAME is a host-side stand-in in host code, not a device address: the address the kernels get comes
// from cudaGetSymbolAddress, asked once per device with that device current (ring_address below).
//
// This file shares nothing with ng.cu / ng_device.cuh but the header: no ng_sim, no Ctl, no allocator.
// =====================================================================================
#include "../../include/ng.h"

#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

namespace {

// The scratch: ring[slot * n_targets + i], slot-major like NG_FIELD_RING.  NG_NOALLOC_MAX_CELLS floats = 16 MiB.
static __device__ __align__(256) float g_noalloc_ring[NG_NOALLOC_MAX_CELLS];
// Records skipped because their target or delay lies outside the sizes of the call (never cleared by a kernel;
// ng_deliver_noalloc_check reads and clears it).
static __device__ unsigned long long g_noalloc_bad;

constexpr int kMaxDevices = 64;
constexpr int kThreads = 256;                    // 8 warps per CTA, one (spike, chunk) item per warp at a time
constexpr int kChunkRecords = 2048;              // records of one item: 16 vector iterations of a warp
constexpr int kChunksPerPass = 8;                // gridDim.y: chunks of one row walked side by side

std::mutex g_mutex;
float* g_ring_ptr[kMaxDevices];                  // device address of g_noalloc_ring, per device (nullptr = not asked yet)
unsigned long long* g_bad_ptr[kMaxDevices];
thread_local char g_err[256] = "";

int32_t fail(int32_t code, const char* fmt, long long a = 0, long long b = 0, long long c = 0) {
    std::snprintf(g_err, sizeof g_err, fmt, a, b, c);
    return code;
}

// Device address of the static ring on the CURRENT device; asked once per device.
int32_t ring_address(float** ring, unsigned long long** bad) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        std::snprintf(g_err, sizeof g_err, "ng_deliver_noalloc: cudaGetDevice: %s", cudaGetErrorString(e));
        return NG_ERR_CUDA;
    }
    if (dev < 0 || dev >= kMaxDevices) return fail(NG_ERR_INVALID_ARG, "ng_deliver_noalloc: device index %lld beyond %lld", dev, kMaxDevices - 1);
    std::lock_guard<std::mutex> lock(g_mutex);
    if (!g_ring_ptr[dev]) {
        float* p = nullptr; unsigned long long* q = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_noalloc_ring);
        if (e == cudaSuccess) e = cudaGetSymbolAddress((void**)&q, g_noalloc_bad);
        if (e != cudaSuccess || !p || !q) {
            std::snprintf(g_err, sizeof g_err, "ng_deliver_noalloc: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));
            return NG_ERR_CUDA;
        }
        g_ring_ptr[dev] = p; g_bad_ptr[dev] = q;
    }
    *ring = g_ring_ptr[dev]; *bad = g_bad_ptr[dev];
    return NG_OK;
}

// out[i] = the input arriving at step n (plane n mod D), and that plane cleared for the spikes that land D steps later.
__global__ void __launch_bounds__(kThreads) noalloc_consume_kernel(float* __restrict__ ring, int N, int slot, float* __restrict__ out) {
    float* plane = ring + (size_t)slot * N;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < N; i += gridDim.x * blockDim.x) {
        out[i] = plane[i];
        plane[i] = 0.f;
    }
}

__device__ __forceinline__ void deliver_one(float* __restrict__ ring, int N, int D, int nmod, int t, float w, int d, unsigned int& bad) {
    if (t < 0) return;                                       // padding record (ng_copy_records)
    if (t >= N || d < 1 || d > D) { bad++; return; }
    int slot = nmod + d; if (slot >= D) slot -= D;
    atomicAdd(ring + (size_t)slot * N + t, w);               // result unused: compiles to red.global.add.f32
}

// One warp per (spike, chunk of kChunkRecords records): blockIdx.y picks the chunk lane of the row, warps stride
// over the spike list.  16-byte loads where the row is laid out as ng_copy_* lays it out (row start and length
// multiples of 4 records, arrays 16-byte aligned: `vec`), scalar loads otherwise.
__global__ void __launch_bounds__(kThreads) noalloc_deliver_kernel(float* __restrict__ ring, unsigned long long* __restrict__ bad_out,
                                                                   const long long* __restrict__ row_off, const int32_t* __restrict__ tgt,
                                                                   const float* __restrict__ w, const uint8_t* __restrict__ dly,
                                                                   int n_sources, const int32_t* __restrict__ spikes, int n_spikes,
                                                                   int N, int D, int nmod, int vec) {
    const int lane = threadIdx.x & 31;
    const int warps = gridDim.x * (kThreads / 32);
    unsigned int bad = 0;
    for (int s = blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5); s < n_spikes; s += warps) {
        const int j = spikes[s];
        if (j < 0 || j >= n_sources) { if (lane == 0 && blockIdx.y == 0) bad++; continue; }
        const long long r0 = row_off[j];
        const long long len = row_off[j + 1] - r0;
        for (long long c0 = (long long)blockIdx.y * kChunkRecords; c0 < len; c0 += (long long)gridDim.y * kChunkRecords) {
            const long long c1 = c0 + kChunkRecords < len ? c0 + kChunkRecords : len;
            if (vec && ((r0 | len) & 3) == 0) {
                for (long long q = c0 + 4 * lane; q < c1; q += 128) {
                    const int4 t = *reinterpret_cast<const int4*>(tgt + r0 + q);
                    const float4 ww = *reinterpret_cast<const float4*>(w + r0 + q);
                    const uchar4 dd = *reinterpret_cast<const uchar4*>(dly + r0 + q);
                    deliver_one(ring, N, D, nmod, t.x, ww.x, dd.x, bad);
                    deliver_one(ring, N, D, nmod, t.y, ww.y, dd.y, bad);
                    deliver_one(ring, N, D, nmod, t.z, ww.z, dd.z, bad);
                    deliver_one(ring, N, D, nmod, t.w, ww.w, dd.w, bad);
                }
            } else {
                for (long long q = c0 + lane; q < c1; q += 32)
                    deliver_one(ring, N, D, nmod, tgt[r0 + q], w[r0 + q], dly[r0 + q], bad);
            }
        }
    }
    if (bad) atomicAdd(bad_out, (unsigned long long)bad);
}

}  // namespace

extern "C" {

const char* ng_noalloc_last_error(void) { return g_err; }

int32_t ng_deliver_noalloc(void* cuda_stream, const int64_t* row_offsets_dev, const int32_t* tgt_dev, const float* w_dev,
                           const uint8_t* delay_dev, int32_t n_sources, const int32_t* spike_ids_dev, int32_t n_spikes,
                           int32_t n_targets, int32_t ring_slots, int64_t step, int32_t reset, float* input_out_dev) {
    g_err[0] = 0;
    if (n_targets < 1 || ring_slots < 1 || ring_slots > 255 || n_sources < 0 || n_spikes < 0 || step < 0)
        return fail(NG_ERR_INVALID_ARG, "ng_deliver_noalloc: need n_targets >= 1, 1 <= ring_slots <= 255, n_sources, n_spikes, step >= 0");
    const long long cells = (long long)n_targets * ring_slots;
    if (cells > (long long)NG_NOALLOC_MAX_CELLS)
        return fail(NG_ERR_INVALID_ARG, "ng_deliver_noalloc: n_targets * ring_slots = %lld cells exceeds the static scratch of "
                                        "NG_NOALLOC_MAX_CELLS = %lld cells (16 MiB); use ng_create / ng_simulate for larger networks",
                    cells, (long long)NG_NOALLOC_MAX_CELLS);
    if (!input_out_dev) return fail(NG_ERR_INVALID_ARG, "ng_deliver_noalloc: input_out_dev is NULL");
    if (n_spikes > 0 && (!row_offsets_dev || !tgt_dev || !w_dev || !delay_dev || !spike_ids_dev))
        return fail(NG_ERR_INVALID_ARG, "ng_deliver_noalloc: NULL connection or spike array with n_spikes = %lld", n_spikes);
    float* ring = nullptr; unsigned long long* bad = nullptr;
    const int32_t rc = ring_address(&ring, &bad);
    if (rc != NG_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaSuccess;
    if (reset) e = cudaMemsetAsync(ring, 0, (size_t)cells * sizeof(float), st);          // the array keeps the last call's contents
    if (e == cudaSuccess) {
        const int nmod = (int)(step % ring_slots);
        int blocks = (n_targets + kThreads - 1) / kThreads; if (blocks > 148 * 8) blocks = 148 * 8;
        noalloc_consume_kernel<<<blocks, kThreads, 0, st>>>(ring, n_targets, nmod, input_out_dev);
        if (n_spikes > 0) {
            const int vec = (((uintptr_t)tgt_dev | (uintptr_t)w_dev) & 15) == 0 && ((uintptr_t)delay_dev & 3) == 0;
            int bx = (n_spikes + kThreads / 32 - 1) / (kThreads / 32); if (bx > 148 * 2) bx = 148 * 2;
            noalloc_deliver_kernel<<<dim3(bx, kChunksPerPass), kThreads, 0, st>>>(ring, bad, (const long long*)row_offsets_dev, tgt_dev, w_dev,
                                                                                 delay_dev, n_sources, spike_ids_dev, n_spikes, n_targets,
                                                                                 ring_slots, nmod, vec);
        }
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        std::snprintf(g_err, sizeof g_err, "ng_deliver_noalloc: %s", cudaGetErrorString(e));
        return NG_ERR_CUDA;
    }
    return NG_OK;
}

int32_t ng_deliver_noalloc_check(void* cuda_stream, int64_t* n_bad_out) {
    g_err[0] = 0;
    float* ring = nullptr; unsigned long long* bad = nullptr;
    const int32_t rc = ring_address(&ring, &bad);
    if (rc != NG_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    unsigned long long v = 0;
    cudaError_t e = cudaMemcpyAsync(&v, bad, sizeof v, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(bad, 0, sizeof v, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) {
        std::snprintf(g_err, sizeof g_err, "ng_deliver_noalloc_check: %s", cudaGetErrorString(e));
        return NG_ERR_CUDA;
    }
    if (n_bad_out) *n_bad_out = (int64_t)v;
    if (v) return fail(NG_ERR_OVERFLOW, "ng_deliver_noalloc: %lld records or spikes outside n_targets / ring_slots / n_sources were skipped", (long long)v);
    return NG_OK;
}

}  // extern "C"

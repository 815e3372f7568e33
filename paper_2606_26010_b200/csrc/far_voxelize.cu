// far_voxelize.cu -- A2 scan downsampling: one representative point per occupied voxel of the scan.
//
// PAPER.md:171 lists downsampling as part of preprocessing without giving the method; reading R2: the
// representative is the LOWEST-INDEX valid point of the voxel and representatives are emitted in ascending
// source index (first-point-per-voxel, so the output is a subset of the input and parity is bit-exact).
//
// Four small kernels, no sort:  (1) find-or-claim the point's key in a scratch open-addressing table and
// atomicMin its index into the voxel's "first index" word;  (2) flag the points that are their voxel's first
// and count flags per tile;  (3) one block scans the tile counts;  (4) stable compaction of the flagged points.
#include <mutex>

#include "far_internal.h"

using namespace far;

namespace far {

constexpr int VTILE = 1024;   // points per tile / threads per block in the flag and scatter passes

struct VoxWs {
    unsigned long long* keys;   // [slots]
    uint32_t* first;            // [slots] lowest point index seen for the key
    uint32_t* slot_of;          // [n]
    uint32_t* tile_off;         // [tiles + 1]
    uint32_t slots, mask;
};

__global__ void __launch_bounds__(256) vox_claim_kernel(VoxWs w, const float* __restrict__ xyz, int64_t n, const int64_t* __restrict__ d_n,
                                                         int stride, float v) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (d_n) n = min(n, *d_n);                  // frame graph: the launch is sized for the largest scan, the count is on the device
    if (i >= n) return;
    const float* p = xyz + i * stride;
    int k[3];
    uint32_t s = NO_SLOT;
    if (voxel_index(p[0], p[1], p[2], v, k)) {
        const unsigned long long key = pack_key(k[0], k[1], k[2]);
        s = hash_key(key) & w.mask;
        for (;;) {   // the scratch table has >= 2n slots, so an empty slot always exists
            unsigned long long cur = *reinterpret_cast<volatile unsigned long long*>(&w.keys[s]);
            if (cur == KEY_EMPTY) cur = atomicCAS(&w.keys[s], KEY_EMPTY, key);
            if (cur == KEY_EMPTY || cur == key) break;
            s = (s + 1) & w.mask;
        }
        atomicMin(&w.first[s], (uint32_t)i);
    }
    w.slot_of[i] = s;
}

__device__ __forceinline__ bool vox_is_first(const VoxWs& w, int64_t i, int64_t n) {
    if (i >= n) return false;
    const uint32_t s = w.slot_of[i];
    return s != NO_SLOT && w.first[s] == (uint32_t)i;
}

__global__ void __launch_bounds__(VTILE) vox_count_kernel(VoxWs w, int64_t n, const int64_t* __restrict__ d_n) {
    __shared__ int s_cnt[VTILE / 32];
    if (d_n) n = min(n, *d_n);
    const int64_t i = (int64_t)blockIdx.x * VTILE + threadIdx.x;
    const unsigned b = __ballot_sync(FULL, vox_is_first(w, i, n));
    if ((threadIdx.x & 31) == 0) s_cnt[threadIdx.x >> 5] = __popc(b);
    __syncthreads();
    if (threadIdx.x < 32) {
        int c = s_cnt[threadIdx.x];
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) c += __shfl_xor_sync(FULL, c, d);
        if (threadIdx.x == 0) w.tile_off[blockIdx.x] = (uint32_t)c;
    }
}

// exclusive scan of the tile counts by one block (tiles = n / 1024: a few thousand at most)
__global__ void __launch_bounds__(1024) vox_scan_kernel(VoxWs w, int tiles, int64_t* n_out) {
    __shared__ uint32_t s_warp[32];
    __shared__ uint32_t s_carry;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int base = 0; base < tiles; base += 1024) {
        const int t = base + threadIdx.x;
        const uint32_t c = t < tiles ? w.tile_off[t] : 0u;
        uint32_t incl = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t o = __shfl_up_sync(FULL, incl, d);
            if (lane >= d) incl += o;
        }
        if (lane == 31) s_warp[wid] = incl;
        __syncthreads();
        if (wid == 0) {
            uint32_t x = s_warp[lane];
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t o = __shfl_up_sync(FULL, x, d);
                if (lane >= d) x += o;
            }
            s_warp[lane] = x;   // inclusive over warps
        }
        __syncthreads();
        const uint32_t warp_excl = wid ? s_warp[wid - 1] : 0u;
        const uint32_t carry = s_carry;
        if (t < tiles) w.tile_off[t] = carry + warp_excl + incl - c;
        __syncthreads();
        if (threadIdx.x == 1023) s_carry = carry + warp_excl + incl;
        __syncthreads();
    }
    if (threadIdx.x == 0) *n_out = (int64_t)s_carry;
}

__global__ void __launch_bounds__(VTILE) vox_scatter_kernel(VoxWs w, const float* __restrict__ xyz, int64_t n, const int64_t* __restrict__ d_n,
                                                             int stride, float* __restrict__ out_xyz, int32_t* __restrict__ out_index) {
    __shared__ int s_cnt[VTILE / 32];
    if (d_n) n = min(n, *d_n);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t i = (int64_t)blockIdx.x * VTILE + threadIdx.x;
    const bool f = vox_is_first(w, i, n);
    const unsigned b = __ballot_sync(FULL, f);
    if (lane == 0) s_cnt[wid] = __popc(b);
    __syncthreads();
    if (wid == 0) {
        const int c = s_cnt[lane];
        int incl = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int o = __shfl_up_sync(FULL, incl, d);
            if (lane >= d) incl += o;
        }
        s_cnt[lane] = incl - c;
    }
    __syncthreads();
    if (f) {
        const int64_t o = (int64_t)w.tile_off[blockIdx.x] + s_cnt[wid] + __popc(b & ((1u << lane) - 1u));
        const float* p = xyz + i * stride;
        out_xyz[3 * o] = p[0]; out_xyz[3 * o + 1] = p[1]; out_xyz[3 * o + 2] = p[2];
        out_index[o] = (int32_t)i;
    }
}

__global__ void zero_i64_kernel(int64_t* p) {
    if (threadIdx.x == 0 && blockIdx.x == 0) *p = 0;
}

static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

}  // namespace far

namespace far {
int voxelize_impl(const float* d_xyz, int64_t n, const int64_t* d_n, int stride, float voxel, float* d_out_xyz, int32_t* d_out_index,
                  int64_t* d_n_out, void* d_workspace, size_t* workspace_bytes, void* stream);
}

extern "C" int far_voxelize(const float* d_xyz, int64_t n, int stride, float voxel, float* d_out_xyz, int32_t* d_out_index,
                            int64_t* d_n_out, void* d_workspace, size_t* workspace_bytes, void* stream) {
    return far::voxelize_impl(d_xyz, n, nullptr, stride, voxel, d_out_xyz, d_out_index, d_n_out, d_workspace, workspace_bytes, stream);
}

// n = min(n, *d_n) if d_n is given (read on the device in stream order)
int far::voxelize_impl(const float* d_xyz, int64_t n, const int64_t* d_n, int stride, float voxel, float* d_out_xyz, int32_t* d_out_index,
                       int64_t* d_n_out, void* d_workspace, size_t* workspace_bytes, void* stream) {
    if (n < 0 || n > (1ll << 30) || (stride != 3 && stride != 4) || !(voxel > 0.f) || !workspace_bytes) return FAR_ERR_ARG;
    uint64_t slots = 64;
    while (slots < 2 * (uint64_t)n) slots <<= 1;
    const int64_t tiles = (n + VTILE - 1) / VTILE;
    const size_t b_keys = align256(slots * 8), b_first = align256(slots * 4), b_slot = align256((size_t)n * 4 + 4),
                 b_tile = align256((size_t)(tiles + 1) * 4);
    const size_t need = b_keys + b_first + b_slot + b_tile;
    if (!d_workspace) { *workspace_bytes = need; return FAR_OK; }
    if (*workspace_bytes < need || !d_n_out || (n > 0 && (!d_xyz || !d_out_xyz || !d_out_index))) return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    if (n == 0) {
        FAR_LAUNCH(zero_i64_kernel, 1, 32, 0, st, d_n_out);
        FAR_CUDA(cudaGetLastError());
        return FAR_OK;
    }
    char* base = static_cast<char*>(d_workspace);
    VoxWs w;
    w.keys = reinterpret_cast<unsigned long long*>(base);
    w.first = reinterpret_cast<uint32_t*>(base + b_keys);
    w.slot_of = reinterpret_cast<uint32_t*>(base + b_keys + b_first);
    w.tile_off = reinterpret_cast<uint32_t*>(base + b_keys + b_first + b_slot);
    w.slots = (uint32_t)slots;
    w.mask = (uint32_t)slots - 1;
    FAR_CUDA(cudaMemsetAsync(base, 0xFF, b_keys + b_first, st));   // keys = empty, first = +inf
    FAR_LAUNCH(vox_claim_kernel, grid_for(n, 256), 256, 0, st, w, d_xyz, n, d_n, stride, voxel);
    FAR_LAUNCH(vox_count_kernel, (int)tiles, VTILE, 0, st, w, n, d_n);
    FAR_LAUNCH(vox_scan_kernel, 1, 1024, 0, st, w, (int)tiles, d_n_out);
    FAR_LAUNCH(vox_scatter_kernel, (int)tiles, VTILE, 0, st, w, d_xyz, n, d_n, stride, d_out_xyz, d_out_index);
    FAR_CUDA(cudaGetLastError());
    return FAR_OK;
}

// ---- far_voxelize_static: the same four kernels with their scratch inside the library ---------------------------
//
// For callers that are not allowed to allocate device memory (see include/far.h: a hard real-time LiDAR callback that
// must stay clear of cudaMalloc's driver locks and device-wide synchronisation, a plug-in whose GPU memory budget is
// owned by its host application, a binding that cannot keep a device buffer between calls).  The scratch far_voxelize
// takes from its caller is here a file-scope device array: it costs FAR_VOXELIZE_STATIC_BYTES on every GPU that loads
// libfar.so, for the life of the process, used or not -- which is why the limit is a modest 262,144 points.
//
// In HOST code the name `g_vox_static` is only a stand-in the runtime registers for the symbol; it is not a device
// address (a kernel handed `g_vox_static` from the host would fault, or on a machine where the GPU can reach host
// memory would quietly scribble over the stand-in).  The address a kernel can use comes from cudaGetSymbolAddress,
// asked once per device with that device current.
namespace far {

constexpr size_t vox_static_need(uint64_t n) {
    uint64_t slots = 64;
    while (slots < 2 * n) slots <<= 1;
    const uint64_t tiles = (n + VTILE - 1) / VTILE;
    return (size_t)(((slots * 8 + 255) & ~255ull) + ((slots * 4 + 255) & ~255ull) + ((n * 4 + 4 + 255) & ~255ull) +
                    (((tiles + 1) * 4 + 255) & ~255ull));
}
static_assert(vox_static_need(FAR_VOXELIZE_STATIC_MAX_POINTS) == FAR_VOXELIZE_STATIC_BYTES,
              "FAR_VOXELIZE_STATIC_BYTES must be the workspace far_voxelize asks for at FAR_VOXELIZE_STATIC_MAX_POINTS");

static __device__ __align__(256) unsigned char g_vox_static[FAR_VOXELIZE_STATIC_BYTES];

constexpr int VOX_STATIC_MAX_DEVICES = 64;
static std::mutex g_vox_static_mu;
static void* g_vox_static_addr[VOX_STATIC_MAX_DEVICES];   // device address of g_vox_static on device i, nullptr = not asked yet

// device address of the scratch on the CURRENT device; the first call on a device asks the runtime, later calls read the cache
static int vox_static_scratch(void** out) {
    int dev = -1;
    FAR_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= VOX_STATIC_MAX_DEVICES) {
        set_cuda_error(cudaErrorInvalidDevice, "far_voxelize_static: supports device ordinals 0..63");
        return FAR_ERR_ARG;
    }
    std::lock_guard<std::mutex> lock(g_vox_static_mu);
    if (!g_vox_static_addr[dev]) {
        void* p = nullptr;
        FAR_CUDA(cudaGetSymbolAddress(&p, g_vox_static));
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255u)) {
            set_cuda_error(cudaErrorInvalidSymbol, "far_voxelize_static: scratch symbol has no 256-byte aligned device address");
            return FAR_ERR_CUDA;
        }
        g_vox_static_addr[dev] = p;
    }
    *out = g_vox_static_addr[dev];
    return FAR_OK;
}

}  // namespace far

extern "C" int far_voxelize_static(const float* d_xyz, int64_t n, int stride, float voxel, float* d_out_xyz, int32_t* d_out_index,
                                   int64_t* d_n_out, void* stream) {
    if (n > (int64_t)FAR_VOXELIZE_STATIC_MAX_POINTS) {
        far::set_cuda_error(cudaErrorInvalidValue,
                            "far_voxelize_static: n exceeds FAR_VOXELIZE_STATIC_MAX_POINTS (262144); use far_voxelize with a caller workspace");
        return FAR_ERR_ARG;
    }
    if (n < 0 || !d_n_out) return FAR_ERR_ARG;
    void* scratch = nullptr;
    const int rc = far::vox_static_scratch(&scratch);   // first call on this device: cudaGetSymbolAddress; afterwards a table read
    if (rc != FAR_OK) return rc;
    // voxelize_impl resets keys / first-index words (cudaMemsetAsync on `stream`) before the claim kernel and writes every
    // slot_of / tile_off word it later reads, so what the previous call left in the array does not matter
    size_t bytes = FAR_VOXELIZE_STATIC_BYTES;
    return far::voxelize_impl(d_xyz, n, nullptr, stride, voxel, d_out_xyz, d_out_index, d_n_out, scratch, &bytes, stream);
}

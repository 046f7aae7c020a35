// aev_static.cu -- aev_pairs_static: the gas-phase cutoff pair search (step (1), SURVEY.md 8(a) rows A1-A2;
// PAPER.md:112 "building neighbor lists") for callers that are not allowed to allocate device memory.
//
// Who that is.  Every other entry point of this library works on an aev_ctx, and aev_create (or a later call
// with larger shapes) obtains the context's workspace with cudaMalloc.  Some hosts cannot do that:
//   - an MD engine or inference server that has handed the whole device to its own pool at start-up, so a
//     cudaMalloc from a plug-in either fails or steals memory the pool believes it owns;
//   - a step loop with a latency budget: cudaMalloc and cudaFree synchronise the device and take a driver lock,
//     which stalls every other stream of the process for the duration;
//   - a component whose device-memory use is audited and fixed when it is linked, so that it may not grow at
//     run time at all.
// For them this file keeps the one piece of working memory the search needs -- the per-atom pair counts that
// turn an unordered search into a sorted, gap-free pair list -- in a file-scope __device__ array.  It is part
// of the loaded library image: every GPU that loads libaev_b200.so carries its 16 KB (4 bytes x
// AEV_STATIC_MAX_ATOMS) until the process exits, and nothing is ever allocated or freed by the call.
//
// Sharing.  There is ONE array per device, used by every call on that device, whichever thread or stream makes
// it.  It still holds whatever the previous call left there.  Nothing in it has to start at zero: pass 0 writes
// deg[0..n) for exactly the n atoms of this call before pass 1 (stream-ordered behind it) reads them, and
// entries beyond n are never read.  Two calls whose kernels can overlap on the GPU (different streams without an
// event between them, or two host threads) race on the array and return wrong pair lists; calls on one stream,
// or ordered by events, are safe.
//
// Product code: shares nothing with oracle/.
#include <mutex>

#include "aev_common.cuh"

using namespace aevb;

namespace {

constexpr int kMaxAtoms = AEV_STATIC_MAX_ATOMS;

// The scratch.  In HOST code `g_pairs_scratch` is only a handle for the runtime's symbol table, not a device
// address: handing it to a kernel would make the kernel fault (or, on a system where the GPU can reach host
// memory, quietly use the wrong bytes).  Host code therefore asks the runtime for the real address once per
// device (scratch_for_device below) and passes that pointer to the kernels.
static __device__ __align__(256) int g_pairs_scratch[kMaxAtoms];      // deg[i], see k_pairs_static

constexpr int kMaxDevices = 64;
std::mutex g_setup_lock;
int *g_scratch_ptr[kMaxDevices];      // device address of g_pairs_scratch on device d; NULL until the set-up ran there

// Set-up, once per device, with that device current (the caller holds a DeviceGuard): resolve the device address
// of the array in this device's copy of the module.  cudaGetSymbolAddress allocates nothing; it may load the
// module on first use, which is why the first call on a device should not come from inside a stream capture.
int scratch_for_device(int device, int **out)
{
    if (device < 0 || device >= kMaxDevices) return AEV_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> hold(g_setup_lock);
    if (!g_scratch_ptr[device]) {
        int major = 0;
        if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device) != cudaSuccess) return AEV_ERR_CUDA;
        if (major != 10) return AEV_ERR_UNSUPPORTED;
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_pairs_scratch);
        if (e != cudaSuccess || !p) return AEV_ERR_CUDA;
        g_scratch_ptr[device] = static_cast<int *>(p);
    }
    *out = g_scratch_ptr[device];
    return AEV_OK;
}

// One warp per atom i, lanes over the partners j > i.  The distance test is the one k_nbr makes
// (d = x_j - x_i in fp32, r2 = fma(dz,dz, fma(dy,dy, dx*dx)), strict r2 < rc*rc), so the pair set is the set
// aev_neighbors + aev_export_pairs give for the same non-periodic system, bit for bit.
//   PASS 0: deg[i] = number of partners j > i of atom i.
//   PASS 1: first slot of atom i = sum of deg[0..i); the pairs of atom i are written from there in ascending j,
//           so the list comes out sorted by (i, j) with no atomics; the warp of the last atom writes the total.
template <int PASS>
__global__ void __launch_bounds__(256)
k_pairs_static(const float *__restrict__ pos, const int32_t *__restrict__ species, int n, float rc2,
               int *__restrict__ deg, int32_t *__restrict__ pairs, long long cap, long long *__restrict__ count_out)
{
    const int lane = threadIdx.x & 31;
    const int i = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (i >= n) return;
    const bool real_i = species ? species[i] >= 0 : true;
    const float xi = pos[3 * i], yi = pos[3 * i + 1], zi = pos[3 * i + 2];
    long long first = 0;
    if (PASS == 1) {
        int s = 0;
        for (int k = lane; k < i; k += 32) s += deg[k];
        first = __reduce_add_sync(0xffffffffu, s);      // < 2^23 pairs for 4096 atoms
    }
    int cnt = 0;
    for (int j0 = i + 1; j0 < n; j0 += 32) {
        const int j = j0 + lane;
        bool hit = false;
        if (real_i && j < n) {
            const bool real_j = species ? species[j] >= 0 : true;
            const float dx = pos[3 * j] - xi, dy = pos[3 * j + 1] - yi, dz = pos[3 * j + 2] - zi;
            const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            hit = real_j && r2 < rc2;
        }
        const unsigned m = __ballot_sync(0xffffffffu, hit);
        if (PASS == 1 && hit) {
            const long long slot = first + cnt + __popc(m & ((1u << lane) - 1u));
            if (slot < cap) { pairs[2 * slot] = i; pairs[2 * slot + 1] = j; }
        }
        cnt += __popc(m);
    }
    if (PASS == 0 && lane == 0) deg[i] = cnt;
    if (PASS == 1 && i == n - 1 && lane == 0) *count_out = first + cnt;
}

}  // namespace

extern "C" int aev_pairs_static(const float *pos, const int32_t *species, int32_t n_atoms, float rc,
                                int32_t *pairs_out, int64_t cap, int64_t *count_out, int32_t device, void *stream)
{
    if ((!pos && n_atoms > 0) || !count_out || n_atoms < 0 || cap < 0 || (cap > 0 && !pairs_out) || !(rc > 0.f))
        return AEV_ERR_INVALID_ARG;
    if (n_atoms > kMaxAtoms) return AEV_ERR_STATIC_LIMIT;      // the array is what it is: nothing to grow
    DeviceGuard guard(device);
    if (!guard.ok()) return AEV_ERR_CUDA;
    int *scratch = nullptr;
    const int rc_setup = scratch_for_device(device, &scratch);
    if (rc_setup != AEV_OK) return rc_setup;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (n_atoms == 0) {
        AEVB_CUDA(cudaMemsetAsync(count_out, 0, sizeof(int64_t), st));
        return AEV_OK;
    }
    int *deg = scratch;
    const float rc2 = rc * rc;
    const int warps = 8, grid = (n_atoms + warps - 1) / warps;
    k_pairs_static<0><<<grid, warps * 32, 0, st>>>(pos, species, n_atoms, rc2, deg, nullptr, 0, nullptr);
    k_pairs_static<1><<<grid, warps * 32, 0, st>>>(pos, species, n_atoms, rc2, deg, pairs_out, (long long)cap,
                                                   reinterpret_cast<long long *>(count_out));
    return cudaGetLastError() == cudaSuccess ? AEV_OK : AEV_ERR_CUDA;
}

// ani_mlp_tc.cu -- per-species MLP forward + transposed chain on the sm_100a tensor cores
// (BASELINE.json:configs[4] "MLP GEMMs in bf16 with fp32 accumulate").
//
// One CTA = one tile of 128 atoms of one species.  Every GEMM of the chain is a tcgen05.mma
// (M = 128 rows, N = layer width, K = 16 per instruction) whose accumulator lives in TMEM:
//   forward  z_l  = h_(l-1) W_l            A = activations (shared memory), B = W_l  [N=out][K=in]
//   backward d_l' = d_(l+1) W_(l+1)^T      A = upstream    (shared memory), B = W^T  [N=in][K=out]
// Activations and weights are fp32 values split into two bf16 operands each (hi + lo); every GEMM
// is hi*hi + lo*hi + hi*lo per K step (the lo*lo term, 2^-18 relative, is dropped).  A network
// whose weights are all bf16-representable (reading G14) has zero weight-lo operands
// and skips the third MMA.  grid.z = model of an ensemble: every model reads the
// same AEV tile and adds its share of the mean energy and of the mean dE/dAEV.  The pre-activations z_l stay resident in TMEM between the forward and the
// backward sweep (CELU' is recomputed from them); bias, CELU, the last (N = 1) layer, the
// energy sum and the bf16 split run in the epilogue, one thread per row (tcgen05.ld 32x32b).
//
// Operand layout in shared memory: K-major, SWIZZLE_128B.  An [R x K] bf16 operand is cut into K blocks of 64
// elements; block kb is R rows of 128 bytes (row r at kb*R*128 + r*128) and inside a row the 16-byte chunk c (8
// elements) sits at chunk position c ^ (r & 7): the 8-row x 128-byte swizzle atoms the tensor core reads without
// bank conflicts (descriptor: SBO = 1024 bytes between 8-row groups, layout type SWIZZLE_128B; one MMA consumes
// K = 16 = 32 bytes, so the start address advances by 32 bytes per K step and by R*128 per block).  Atoms are
// 1024-byte aligned.  The unswizzled "core matrix" layout of round 1 ran the MMAs at 2.8 x their floor.
#include <cuda_bf16.h>
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <memory>
#include <vector>

#include "aev_common.cuh"

using namespace aevb;

namespace {

// -DAEVB_TC_TIMING: CTA (0,0) prints the clock64 offsets of its phase boundaries (debug builds only)
#ifdef AEVB_TC_TIMING
#define TC_STAMP(i) do { if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) ts_[i] = clock64() - t0_; } while (0)
#else
#define TC_STAMP(i) do { } while (0)
#endif

constexpr int kTM = 128;              // rows (atoms) per tile = MMA M
constexpr int kTcGroups = 8;          // warpgroups per CTA: group g takes the 8-column chunks g, g+8, ... in the epilogues
constexpr int kTcThreads = kTM * kTcGroups;
constexpr int kKC = 64;               // K chunk of the first layer (AEV columns per stage)
constexpr int kActBytes = 98304;      // activation operand: hi | lo, each up to 3 K blocks (K <= 192) of 128 rows x 128 bytes
constexpr int kActHalf = kActBytes / 2;
constexpr int kWBufBytes = 49152;     // one weight buffer (two of them, ping-pong): e.g. 3 K blocks x 128 rows x 128 bytes
constexpr int kABlk = kTM * 128;      // bytes of one K block of the activation operand
constexpr int kTcSmem = kActBytes + 2 * kWBufBytes + 1024;

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(void *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_wait(void *bar, unsigned parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void proxy_fence() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// D[tmem] (+)= A[smem] * B[smem]; single thread issues on behalf of the CTA.
__device__ __forceinline__ void umma_bf16(unsigned d_tmem, unsigned long long a_desc, unsigned long long b_desc,
                                          unsigned idesc, unsigned accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// arrive on an mbarrier once every MMA issued so far by this thread has completed
__device__ __forceinline__ void umma_commit(void *bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void tmem_ld8(unsigned taddr, float *v)      // no wait: pair with tmem_wait()
{
    unsigned r[8];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr)
                 : "memory");
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = __uint_as_float(r[k]);
}
__device__ __forceinline__ void tmem_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// shared-memory matrix descriptor: K-major, SWIZZLE_128B (layout type 2 in bits 61-63), SBO = 1024 bytes, version 1
// (sm_100); the leading-dimension offset is not used by swizzled K-major operands
__device__ __forceinline__ unsigned long long smem_desc(unsigned addr)
{
    return (unsigned long long)((addr >> 4) & 0x3FFF) | ((unsigned long long)(1024 >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// byte offset of the 16-byte chunk c (8 elements along K) of row r in an operand of R rows
__device__ __forceinline__ unsigned sw_off(int r, int c, int R)
{
    return (unsigned)((c >> 3) * R * 128 + r * 128 + (((c & 7) ^ (r & 7)) << 4));
}
// instruction descriptor: kind::f16, A = B = bf16 (K-major), D = f32, M = 128, N = n
__device__ __forceinline__ unsigned instr_desc(int n)
{
    return (1u << 4) | (1u << 7) | (1u << 10) | ((unsigned)(n >> 3) << 17) | ((unsigned)(kTM >> 4) << 24);
}

__device__ __forceinline__ void cp_async16_tc(void *smem_dst, const void *gsrc)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all_tc() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// 32-byte global accesses (one request per thread: rows are 1.5 KB apart, every lane its own sector)
__device__ __forceinline__ void ldg256(const float *p, float *v)
{
    asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7])
                 : "l"(p));
}
// 16-byte vector reduction (sm_90+): four fp32 adds in one request
__device__ __forceinline__ void red_add_v4(float *p, const float *v)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(p), "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]) : "memory");
}
__device__ __forceinline__ void stg256(float *p, const float *v)
{
    asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "f"(v[0]), "f"(v[1]), "f"(v[2]),
                 "f"(v[3]), "f"(v[4]), "f"(v[5]), "f"(v[6]), "f"(v[7])
                 : "memory");
}

// fp32 x8 -> bf16 hi x8 (16 bytes) and bf16 lo x8 (residual)
__device__ __forceinline__ void split8(const float *v, uint4 &hi, uint4 &lo)
{
    unsigned h[4], l[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const __nv_bfloat162 hh = __floats2bfloat162_rn(v[2 * k], v[2 * k + 1]);
        h[k] = *reinterpret_cast<const unsigned *>(&hh);
        // bf16 -> fp32 is a 16-bit shift
        const float f0 = __uint_as_float(h[k] << 16), f1 = __uint_as_float(h[k] & 0xffff0000u);
        const __nv_bfloat162 ll = __floats2bfloat162_rn(v[2 * k] - f0, v[2 * k + 1] - f1);
        l[k] = *reinterpret_cast<const unsigned *>(&ll);
    }
    hi = make_uint4(h[0], h[1], h[2], h[3]);
    lo = make_uint4(l[0], l[1], l[2], l[3]);
}

__device__ __forceinline__ float celu_tc(float x, float alpha, float inv_alpha)
{
    return x > 0.f ? x : alpha * (__expf(x * inv_alpha) - 1.0f);
}
__device__ __forceinline__ float dcelu_tc(float x, float inv_alpha) { return x > 0.f ? 1.0f : __expf(x * inv_alpha); }

struct TcNetDev {
    int loaded, nh;                      // nh = hidden layers (1..3); layer l maps dims[l] -> dims[l+1]
    int need_lo;                         // some hidden-layer weight is not bf16-representable: third MMA per K step
    float alpha;                         // CELU alpha
    int dims[kMaxMlpLayers + 1];         // dims[0] = L, dims[1..nh] hidden widths, dims[nh+1] = 1
    const __nv_bfloat16 *wf[3];          // forward operand of layer l:  hi [K/8][N][8] | lo, K = dims[l],   N = dims[l+1]
    const __nv_bfloat16 *wb[3];          // backward operand of layer l: hi [K/8][N][8] | lo, K = dims[l+1], N = dims[l]
    const float *bias[3];                // bias of layer l (width dims[l+1])
    const float *wlast;                  // last layer weights [dims[nh]]
    float blast;
    int zoff[3];                         // TMEM column of z_(l+1) = output of layer l
};
struct TcAll { TcNetDev net[kMaxModels][kMaxS]; };

__global__ void __launch_bounds__(kTcThreads, 1)
k_mlp_tc(const TcAll *__restrict__ Mg, int n_models, int L, int n_total, int n_atoms,
         const int *__restrict__ sp_rows, const int *__restrict__ sp_count, const float *__restrict__ aev,
         float *__restrict__ grad, double *__restrict__ energy, int *__restrict__ err)
{
    extern __shared__ __align__(1024) unsigned char sm[];
    __shared__ int s_row[kTM];
    pdl_trigger();
    // everything up to the first AEV load runs before griddepcontrol.wait: the species partition (k_group) was
    // complete before k_bin started, the weights are static, TMEM and barriers are this CTA's own
    const int s = blockIdx.y;
    const int rows = sp_count[s];
    const int r0 = blockIdx.x * kTM;
    // (a CTA that leaves early still passes griddepcontrol.wait: completion of this grid must imply completion
    //  of everything before it in the launch chain - aev_common.cuh)
    if (r0 >= rows) { pdl_wait(); return; }
    __shared__ TcNetDev N;
    if (threadIdx.x < sizeof(TcNetDev) / 4)
        reinterpret_cast<int *>(&N)[threadIdx.x] = reinterpret_cast<const int *>(&Mg->net[blockIdx.z][s])[threadIdx.x];
    __syncthreads();
    if (!N.loaded) { if (threadIdx.x == 0) atomicOr(err, kErrBitState); pdl_wait(); return; }
    const int tid = threadIdx.x, wid = tid >> 5;
    const int row = tid & (kTM - 1), grp = tid >> 7;     // epilogue: thread = (row, column group)
    const float alpha = N.alpha, inv_alpha = 1.0f / alpha;
    const float inv_m = 1.0f / (float)n_models;
    const int nh = N.nh;
    const bool need_lo = N.need_lo != 0;

    unsigned char *act = sm;
    unsigned char *wbuf[2] = {sm + kActBytes, sm + kActBytes + kWBufBytes};
    unsigned long long *bar = reinterpret_cast<unsigned long long *>(sm + kActBytes + 2 * kWBufBytes);
    unsigned *tmem_slot = reinterpret_cast<unsigned *>(bar + 4);

    if (tid == 0) {
        mbar_init(&bar[0], 1); mbar_init(&bar[1], 1); mbar_init(&bar[2], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (wid == 0) {      // one warp owns the TMEM allocation (all 512 columns: one CTA per SM)
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (tid < kTM) s_row[tid] = (r0 + tid < rows) ? sp_rows[(size_t)s * n_total + r0 + tid] : -1;
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const unsigned tmem = *tmem_slot;
    const unsigned tlane = tmem + ((unsigned)((wid & 3) * 32) << 16);   // this warp's quarter of the 128 lanes
    const int my_row = s_row[row];
    unsigned ph0 = 0, ph1 = 0, ph2 = 0;
#ifdef AEVB_TC_TIMING
    __shared__ long long ts_[8];
    const long long t0_ = clock64();
#endif
    TC_STAMP(0);

    // ------------------------------------------------------------------ layer 0, K in chunks
    {
        const int K0 = N.dims[0], N1 = N.dims[1];
        const unsigned idesc = instr_desc(N1);
        const int nkc = (K0 + kKC - 1) / kKC;
        struct F8 { float v[8]; };
        // this thread's k-chunk (8 AEV columns) of stages kc and kc+1 travel in registers
        auto load_a = [&](int kc) -> F8 {
            F8 x;
            const int col = kc * kKC + grp * 8;
            if (my_row >= 0 && col < K0) {
                ldg256(aev + (size_t)my_row * L + col, x.v);
            } else {
#pragma unroll
                for (int k = 0; k < 8; ++k) x.v[k] = 0.f;
            }
            return x;
        };
        auto load_w0 = [&](int kc) {      // stage kc of W_0: a contiguous block of the [K/8][N][8] operand
            const int kw = min(kKC, K0 - kc * kKC);
            // K block kc of the packed operand: N1 rows x 128 bytes, already swizzled (a partial last block is zero-padded)
            const unsigned char *src = reinterpret_cast<const unsigned char *>(N.wf[0]) + (size_t)kc * N1 * 128;
            unsigned char *dst = wbuf[kc & 1];
            const int pieces = 8 * N1;
            (void)kw;
            for (int t = tid; t < pieces; t += kTcThreads) cp_async16_tc(dst + t * 16, src + (size_t)t * 16);
            if (need_lo) {      // residual operand: second half of the stage buffer
                const unsigned char *srcl = src + (size_t)((K0 + 63) / 64) * N1 * 128;
                for (int t = tid; t < pieces; t += kTcThreads)
                    cp_async16_tc(dst + kWBufBytes / 2 + t * 16, srcl + (size_t)t * 16);
            }
        };
        load_w0(0);
        pdl_wait();              // the AEV rows (k_aev) are complete
        F8 x0 = load_a(0), x1 = load_a(1);
        for (int kc = 0; kc < nkc; ++kc) {
            const int b = kc & 1;
            const int kw = min(kKC, K0 - kc * kKC);
            unsigned char *abuf = act + b * 32768;         // hi at +0, lo at +16384
            // (the MMAs that read abuf / wbuf[b] two stages ago were waited for in the previous iteration)
            if (grp < kw / 8) {          // this thread's k-chunk of the stage: columns kc*64 + grp*8 .. +7
                uint4 hi, lo;
                split8(x0.v, hi, lo);
                *reinterpret_cast<uint4 *>(abuf + sw_off(row, grp, kTM)) = hi;
                *reinterpret_cast<uint4 *>(abuf + 16384 + sw_off(row, grp, kTM)) = lo;
            }
            x0 = x1;
            x1 = load_a(kc + 2);         // two stages ahead (zeros past the last stage)
            cp_async_wait_all_tc();      // W_0 stage kc was requested one stage ago
            proxy_fence();
            tc_fence_before();
            __syncthreads();
            if (tid == 0) {
                tc_fence_after();
                const unsigned a_hi = smem_u32(abuf), a_lo = a_hi + 16384, b_a = smem_u32(wbuf[b]);
                for (int ks = 0; ks < kw / 16; ++ks) {
                    const unsigned long long bd = smem_desc(b_a + ks * 32);
                    umma_bf16(tmem + N.zoff[0], smem_desc(a_hi + ks * 32), bd, idesc, (kc | ks) != 0);
                    umma_bf16(tmem + N.zoff[0], smem_desc(a_lo + ks * 32), bd, idesc, 1u);
                    if (need_lo)
                        umma_bf16(tmem + N.zoff[0], smem_desc(a_hi + ks * 32), smem_desc(b_a + kWBufBytes / 2 + ks * 32), idesc, 1u);
                }
                umma_commit(&bar[b]);
            }
            if (kc + 1 < nkc) {
                // the other buffer pair is free once the MMAs of stage kc-1 are done; then prefetch W_0 stage kc+1
                if (kc >= 1) {
                    if (b == 1) { mbar_wait(&bar[0], ph0); ph0 ^= 1; } else { mbar_wait(&bar[1], ph1); ph1 ^= 1; }
                }
                load_w0(kc + 1);
            }
        }
        // drain the commits not waited for above: stage nkc-2 (if any), then stage nkc-1
        if (nkc >= 2) {
            if (((nkc - 2) & 1) == 0) { mbar_wait(&bar[0], ph0); ph0 ^= 1; } else { mbar_wait(&bar[1], ph1); ph1 ^= 1; }
        }
        if (((nkc - 1) & 1) == 0) { mbar_wait(&bar[0], ph0); ph0 ^= 1; } else { mbar_wait(&bar[1], ph1); ph1 ^= 1; }
        tc_fence_after();
    }

    TC_STAMP(1);
    // whole-layer weight operand -> shared memory (contiguous [K/8][N][8] block; the residual operand right behind it)
    auto load_w = [&](const __nv_bfloat16 *w, int K, int Nn, unsigned char *dst) {
        const unsigned char *src = reinterpret_cast<const unsigned char *>(w);
        const int pieces = ((K + 63) / 64) * Nn * 8 * (need_lo ? 2 : 1);      // hi | lo are adjacent in global memory too
        for (int t = tid; t < pieces; t += kTcThreads) cp_async16_tc(dst + t * 16, src + (size_t)t * 16);
    };
    // D[tmem + dcol] = act[128 x K] (hi + lo) * B[Nn x K]^T (hi [+ lo behind the hi blocks]), issued by one thread,
    // completion on bar[2]
    auto gemm = [&](int K, int Nn, const unsigned char *wsm, unsigned dcol) {
        if (tid == 0) {
            tc_fence_after();
            const unsigned a_hi = smem_u32(act), a_lo = a_hi + kActHalf, b_a = smem_u32(wsm);
            const unsigned idesc = instr_desc(Nn);
            const unsigned b_lo = b_a + ((K + 63) / 64) * Nn * 128;
            for (int ks = 0; ks < K / 16; ++ks) {
                const unsigned ao = (ks >> 2) * kABlk + (ks & 3) * 32, bo = (ks >> 2) * Nn * 128 + (ks & 3) * 32;
                const unsigned long long bd = smem_desc(b_a + bo);
                umma_bf16(tmem + dcol, smem_desc(a_hi + ao), bd, idesc, ks != 0);
                umma_bf16(tmem + dcol, smem_desc(a_lo + ao), bd, idesc, 1u);
                if (need_lo) umma_bf16(tmem + dcol, smem_desc(a_hi + ao), smem_desc(b_lo + bo), idesc, 1u);
            }
            umma_commit(&bar[2]);
        }
    };
    auto wait_gemm = [&]() {
        mbar_wait(&bar[2], ph2);
        ph2 ^= 1;
        tc_fence_after();
    };
    // 8 fp32 values of this thread's row -> operand k-chunk c (columns 8c..8c+7), hi and lo
    auto put8 = [&](const float *v, int c) {
        uint4 hi, lo;
        split8(v, hi, lo);
        *reinterpret_cast<uint4 *>(act + sw_off(row, c, kTM)) = hi;
        *reinterpret_cast<uint4 *>(act + kActHalf + sw_off(row, c, kTM)) = lo;
    };
    auto sync_for_mma = [&]() {      // generic-proxy writes + cp.async data visible to the tensor core
        cp_async_wait_all_tc();
        proxy_fence();
        tc_fence_before();
        __syncthreads();
    };
    constexpr int kMaxC = 3;         // 8-column chunks per thread in a hidden-layer epilogue (width <= 160... 192)

    // ------------------------------------------------------------------ forward, layers 1 .. nh-1
    int wsel = 0;
    for (int l = 1; l <= nh; ++l) {
        // z_l (output of layer l-1) is complete in TMEM at zoff[l-1]
        const int Nl = N.dims[l], ncl = Nl >> 3;
        const float *bl = N.bias[l - 1];
        // (every earlier GEMM has completed here, so with residual operands - up to 80 KB, both buffers - the
        //  operand always starts at wbuf[0])
        if (need_lo) wsel = 0;
        if (l < nh) load_w(N.wf[l], Nl, N.dims[l + 1], wbuf[wsel]);               // overlaps the epilogue below
        else if (nh >= 2) load_w(N.wb[nh - 1], Nl, N.dims[nh - 1], wbuf[wsel]);
        float v[kMaxC][8];
#pragma unroll
        for (int i = 0; i < kMaxC; ++i) {
            const int c = grp + i * kTcGroups;
            if (c < ncl) tmem_ld8(tlane + N.zoff[l - 1] + c * 8, v[i]);
        }
        tmem_wait();
        float e = 0.f;
#pragma unroll
        for (int i = 0; i < kMaxC; ++i) {
            const int c = grp + i * kTcGroups;
            if (c < ncl) {
                const float4 b0 = __ldg(reinterpret_cast<const float4 *>(bl + c * 8));
                const float4 b1 = __ldg(reinterpret_cast<const float4 *>(bl + c * 8) + 1);
                const float bb[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
                if (l < nh) {
#pragma unroll
                    for (int k = 0; k < 8; ++k) v[i][k] = celu_tc(v[i][k] + bb[k], alpha, inv_alpha);
                } else {
                    // last hidden layer: energy (the N = 1 layer, CUDA cores) and d_nh = w_last * CELU'(z)
                    const float4 w0 = __ldg(reinterpret_cast<const float4 *>(N.wlast + c * 8));
                    const float4 w1 = __ldg(reinterpret_cast<const float4 *>(N.wlast + c * 8) + 1);
                    const float ww[8] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
#pragma unroll
                    for (int k = 0; k < 8; ++k) {
                        const float z = v[i][k] + bb[k];
                        e = fmaf(celu_tc(z, alpha, inv_alpha), ww[k], e);
                        v[i][k] = ww[k] * dcelu_tc(z, inv_alpha);
                    }
                }
                put8(v[i], c);
            }
        }
        if (l < nh) {
            sync_for_mma();
            gemm(Nl, N.dims[l + 1], wbuf[wsel], N.zoff[l]);
            wsel ^= 1;
            wait_gemm();
        } else {
            // energy: one fp64 atomic per warp when its rows belong to one system (the usual case)
            double ed = my_row >= 0 ? ((double)e + (grp == 0 ? (double)N.blast : 0.0)) * (double)inv_m : 0.0;
            const int bsys = my_row >= 0 ? my_row / n_atoms : -1;
            const unsigned have = __ballot_sync(0xffffffffu, my_row >= 0);
            if (have) {
                const int b0 = __shfl_sync(0xffffffffu, bsys, __ffs(have) - 1);
                if (__all_sync(0xffffffffu, bsys == b0 || bsys < 0)) {
#pragma unroll
                    for (int o = 16; o >= 1; o >>= 1) ed += __shfl_xor_sync(0xffffffffu, ed, o);
                    if ((tid & 31) == 0) atomicAdd(&energy[b0], ed);
                } else if (my_row >= 0) {
                    atomicAdd(&energy[bsys], ed);
                }
            }
        }
    }

    TC_STAMP(2);
    // ------------------------------------------------------------------ backward, layers nh-1 .. 1
    for (int l = nh - 1; l >= 1; --l) {
        // act holds d_(l+1) [128 x dims[l+1]]; wbuf[wsel] holds (or is receiving) the W_l^T operand
        const int Kb = N.dims[l + 1], Nb = N.dims[l], ncl = Nb >> 3;
        const unsigned dcol = N.zoff[l];                   // z_(l+1) is dead: reuse its columns
        sync_for_mma();
        gemm(Kb, Nb, wbuf[wsel], dcol);
        if (!need_lo) {
            wsel ^= 1;
            if (l >= 2) load_w(N.wb[l - 1], Nb, N.dims[l - 1], wbuf[wsel]);   // next operand while the MMAs run
            wait_gemm();
        } else {      // residual operands span both buffers: the next operand follows the GEMM
            wait_gemm();
            if (l >= 2) load_w(N.wb[l - 1], Nb, N.dims[l - 1], wbuf[0]);
        }
        const float *bl = N.bias[l - 1];
#pragma unroll
        for (int i = 0; i < kMaxC; ++i) {
            const int c = grp + i * kTcGroups;
            if (c < ncl) {
                float d[8], z[8];
                tmem_ld8(tlane + dcol + c * 8, d);
                tmem_ld8(tlane + N.zoff[l - 1] + c * 8, z);
                const float4 b0 = __ldg(reinterpret_cast<const float4 *>(bl + c * 8));
                const float4 b1 = __ldg(reinterpret_cast<const float4 *>(bl + c * 8) + 1);
                const float bb[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
                tmem_wait();
#pragma unroll
                for (int k = 0; k < 8; ++k) d[k] *= dcelu_tc(z[k] + bb[k], inv_alpha);
                put8(d, c);
            }
        }
    }

    TC_STAMP(3);
    // ------------------------------------------------------------------ d_0 = d_1 W_0^T, N = L in chunks of CW
    {
        const int Kb = N.dims[1];
        const int CW = need_lo ? 64 : 128;       // a chunk's hi (+ lo) operand fits one 48 KB buffer
        const int nch = (L + CW - 1) / CW;
        const int nkb = (Kb + 63) / 64;
        const size_t lo_off = (size_t)nkb * L * 128;
        if (need_lo) wsel = 0;
        auto load_chunk = [&](int j, unsigned char *dst) {
            const int n0 = j * CW, nw = min(CW, L - n0);
            const unsigned char *src = reinterpret_cast<const unsigned char *>(N.wb[0]);
            const int per = nw * 8, pieces = nkb * per;      // K block kb of the chunk: rows n0 .. n0+nw-1, 128 bytes each
            for (int t = tid; t < pieces; t += kTcThreads) {
                const int kb = t / per, q = t - kb * per;
                const size_t so = ((size_t)kb * L + n0) * 128 + (size_t)q * 16;
                cp_async16_tc(dst + t * 16, src + so);
                if (need_lo) cp_async16_tc(dst + pieces * 16 + t * 16, src + lo_off + so);
            }
        };
        // accumulators alternate between two TMEM slots (every z is dead by now): chunk j at column (j & 1) * 128
        load_chunk(0, wbuf[wsel]);
        sync_for_mma();
        gemm(Kb, min(CW, L), wbuf[wsel], 0u);
        for (int j = 0; j < nch; ++j) {
            const int n0 = j * CW, nw = min(CW, L - n0);
            const unsigned slot = (unsigned)(j & 1) * 128u;
            if (j + 1 < nch) load_chunk(j + 1, wbuf[wsel ^ 1]);
            wait_gemm();
            if (j + 1 < nch) {
                const int nw1 = min(CW, L - (j + 1) * CW);
                sync_for_mma();
                gemm(Kb, nw1, wbuf[wsel ^ 1], slot ^ 128u);
                wsel ^= 1;
            }
            // tcgen05.ld is warp-collective: rows without an atom take part, only the store is skipped
            float *dst = grad + (size_t)(my_row >= 0 ? my_row : 0) * L + n0;
            float v[2][8];
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const int c = grp + i * kTcGroups;
                if (c * 8 < nw) tmem_ld8(tlane + slot + c * 8, v[i]);
            }
            tmem_wait();
            // the epilogue of chunk j must have read its slot before the GEMM of chunk j+2 overwrites it: that GEMM is
            // issued after the next iteration's sync_for_mma (a CTA-wide barrier behind this read)
            tc_fence_before();
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const int c = grp + i * kTcGroups;
                if (c * 8 < nw && my_row >= 0) {
                    if (n_models == 1) {
                        stg256(dst + c * 8, v[i]);
                    } else {      // mean over the ensemble: grad was zeroed before the launch chain
#pragma unroll
                        for (int k = 0; k < 8; ++k) v[i][k] *= inv_m;
                        red_add_v4(dst + c * 8, v[i]);
                        red_add_v4(dst + c * 8 + 4, v[i] + 4);
                    }
                }
            }
        }
    }

    TC_STAMP(4);
#ifdef AEVB_TC_TIMING
    if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0)
        printf("TC %lld %lld %lld %lld %lld\n", ts_[0], ts_[1], ts_[2], ts_[3], ts_[4]);
#endif
    // ------------------------------------------------------------------ teardown
    tc_fence_before();
    __syncthreads();
    if (wid == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
}


}  // namespace

namespace aevb {

// Shapes the tensor-core kernel covers (everything else runs the fp32 CUDA-core kernel):
// 1..3 hidden layers of width 16..160 (multiples of 16), L a multiple of 16, the weight operand of
// every inner layer within the shared-memory buffers (40 KB; 80 KB hi + lo for weights that are not
// bf16-representable), z_l and the backward accumulators within 512 TMEM columns.
bool mlp_tc_eligible(const MlpNet &n, int L)
{
    const int nh = n.n_layers - 1;
    if (nh < 1 || nh > 3) return false;
    if (L % 16 || L > 4096 || n.dims[0] != L) return false;
    const int wlim = n.bf16_exact ? kWBufBytes : 2 * kWBufBytes, per = n.bf16_exact ? 1 : 2;
    int off = 0;
    for (int l = 1; l <= nh; ++l) {
        if (n.dims[l] % 16 || n.dims[l] < 16 || n.dims[l] > 160) return false;
        off += n.dims[l];
    }
    if (off > 512) return false;
    if (n.dims[1] * 128 > kWBufBytes / 2) return false;                       // one K block of W_0 (hi | lo halves)
    for (int l = 1; l < nh; ++l) {                                            // inner layers, forward and backward operand
        if (((n.dims[l] + 63) / 64) * n.dims[l + 1] * 128 * per > wlim) return false;
        if (((n.dims[l + 1] + 63) / 64) * n.dims[l] * 128 * per > wlim) return false;
    }
    if (((n.dims[1] + 63) / 64) * 128 * 128 > kWBufBytes) return false;         // a 128- (64-) column chunk of W_0^T
    // backward accumulator of layer l reuses the columns from z_(l+1) on
    int zo = 0;
    for (int l = 1; l < nh; ++l) {
        zo += n.dims[l];                       // = zoff of z_(l+1)
        if (zo + n.dims[l] > 512) return false;
    }
    return true;
}

// Builds the device table of tensor-core operands; called whenever a network is (re)loaded.  Syncs.
int mlp_tc_upload(aev_ctx *c)
{
    const int S = c->dp.S;
    // 9 KB, built on the heap per call: two contexts may load networks from two host threads at once
    std::unique_ptr<TcAll> Mp(new TcAll);
    TcAll &M = *Mp;
    memset(&M, 0, sizeof(M));
    for (int m = 0; m < c->n_models; ++m)
        for (int s = 0; s < S; ++s) {
            const MlpNet &n = c->nets[m][s];
            TcNetDev &d = M.net[m][s];
            d.loaded = n.loaded;
            if (!n.loaded || !n.tc_ok) continue;
            d.nh = n.n_layers - 1;
            d.need_lo = n.bf16_exact ? 0 : 1;
            d.alpha = n.alpha;
            for (int l = 0; l <= n.n_layers; ++l) d.dims[l] = n.dims[l];
            int off = 0;
            for (int l = 0; l < d.nh; ++l) {
                d.wf[l] = static_cast<const __nv_bfloat16 *>(n.w_fwd[l]);
                d.wb[l] = static_cast<const __nv_bfloat16 *>(n.w_bwd[l]);
                d.bias[l] = n.bias[l];
                d.zoff[l] = off;
                off += n.dims[l + 1];
            }
            d.wlast = n.w_f32[d.nh];
            d.blast = n.b_last;
        }
    if (!c->tc_dev) AEVB_CUDA(cudaMalloc(&c->tc_dev, sizeof(TcAll)));
    AEVB_CUDA(cudaMemcpy(c->tc_dev, &M, sizeof(TcAll), cudaMemcpyHostToDevice));
    return AEV_OK;
}

int mlp_tc_forward_backward(aev_ctx *c, int n_total, int n_atoms, const float *aev, float *grad_aev,
                            double *energy_out, cudaStream_t st)
{
    const int S = c->dp.S, L = c->dp.L;
    if (!c->tc_dev) return AEV_ERR_STATE;
    if (!c->tc_smem_optin) {
        AEVB_CUDA(cudaFuncSetAttribute(k_mlp_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, kTcSmem));
        c->tc_smem_optin = 1;
    }
    dim3 grid((n_total + kTM - 1) / kTM, S, c->n_models);
    if ((c->hp.flags & AEV_FLAG_DETERMINISTIC) && c->n_models > 1) {
        // bit-reproducible mean dE/dAEV: one launch per model, so the fp32 REDs of the models land on every element in
        // model order (within one launch each element is added to once); grid.z = 1 and the table pointer advanced
        // to model m's row, so that blockIdx.z = 0 addresses it
        grid.z = 1;
        for (int m = 0; m < c->n_models; ++m) {
            const TcAll *row = reinterpret_cast<const TcAll *>(static_cast<const TcAll *>(c->tc_dev)->net + m);
            launch_pdl(k_mlp_tc, grid, dim3(kTcThreads), (size_t)kTcSmem, st, row, c->n_models, L, n_total, n_atoms,
                       (const int *)c->sp_rows, (const int *)c->sp_count, aev, grad_aev, energy_out, c->ws.err);
        }
        c->launches += c->n_models - 1;
        return cudaGetLastError() == cudaSuccess ? AEV_OK : AEV_ERR_CUDA;
    }
    launch_pdl(k_mlp_tc, grid, dim3(kTcThreads), (size_t)kTcSmem, st, static_cast<const TcAll *>(c->tc_dev), c->n_models, L,
               n_total, n_atoms, (const int *)c->sp_rows, (const int *)c->sp_count, aev, grad_aev, energy_out, c->ws.err);
    return cudaGetLastError() == cudaSuccess ? AEV_OK : AEV_ERR_CUDA;
}

// Host-side packing of one layer W[in][out] (row-major) into the two swizzled K-major operand layouts (see the file
// header), each as the bf16 hi parts followed by the bf16 residuals (w - hi) in the same layout:
//   forward  operand B[n = out][k = in]:  K blocks of 64 inputs,  N_out rows of 128 bytes per block
//   backward operand B[n = in][k = out]:  K blocks of 64 outputs, K_in  rows of 128 bytes per block
void mlp_tc_pack(const float *w, int K_in, int N_out, std::vector<__nv_bfloat16> &fwd, std::vector<__nv_bfloat16> &bwd,
                 bool *exact)
{
    auto idx = [](int row, int k, int rows) -> size_t {      // element index of (row, k) in an operand of `rows` rows
        const int kb = k >> 6, c = (k & 63) >> 3;
        return (size_t)kb * rows * 64 + (size_t)row * 64 + (size_t)((c ^ (row & 7)) << 3) + (k & 7);
    };
    const size_t nf = (size_t)((K_in + 63) / 64) * N_out * 64, nb = (size_t)((N_out + 63) / 64) * K_in * 64;
    fwd.assign(2 * nf, __float2bfloat16_rn(0.f));
    bwd.assign(2 * nb, __float2bfloat16_rn(0.f));
    bool ex = true;
    for (int k = 0; k < K_in; ++k)
        for (int o = 0; o < N_out; ++o) {
            const float v = w[(size_t)k * N_out + o];
            const __nv_bfloat16 b = __float2bfloat16_rn(v);
            const __nv_bfloat16 r = __float2bfloat16_rn(v - __bfloat162float(b));
            if (__bfloat162float(b) != v) ex = false;
            const size_t fi = idx(o, k, N_out), bi = idx(k, o, K_in);
            fwd[fi] = b; fwd[nf + fi] = r;
            bwd[bi] = b; bwd[nb + bi] = r;
        }
    *exact = ex;
}

}  // namespace aevb

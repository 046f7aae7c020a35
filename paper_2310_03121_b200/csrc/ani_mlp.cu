// ani_mlp.cu -- species-batched per-atom networks:
//   z^l = h^(l-1) W^l + b^l,  h^l = CELU_alpha(z^l) (hidden), last layer linear, E = sum_i E_i,
//   and the transposed chain dE/dAEV (BASELINE.json:configs[4]; DESIGN.md section 3 step 6).
#include <cuda_bf16.h>
#include <math.h>
#include <string.h>

#include <memory>
#include <vector>

#include "aev_common.cuh"

using namespace aevb;

namespace {

struct MlpDev {
    int loaded, n_layers;
    int dims[kMaxMlpLayers + 1];
    const float *w[kMaxMlpLayers];
    const float *wt[kMaxMlpLayers];
    const float *b[kMaxMlpLayers];
    float alpha;
};
struct MlpAll { MlpDev net[kMaxModels][kMaxS]; };

// Partition of the caller's atoms by species: sp_rows[s][0..sp_count[s]).  Slots are handed out
// with one warp-aggregated atomic per (warp, species); the order inside a species is arbitrary
// (rows are independent in the GEMMs; the energy sum is an fp64 atomic either way).
// sp_count must be zero on entry.
__global__ void __launch_bounds__(256) k_group(int n_total, int S, const int32_t *__restrict__ species,
                                               int *__restrict__ sp_rows, int *__restrict__ sp_count,
                                               double *__restrict__ energy, int batch)
{
    const int a = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31;
    if (blockIdx.x == 0)
        for (int b = threadIdx.x; b < batch; b += blockDim.x) energy[b] = 0.0;
    const int sp = a < n_total ? species[a] : -1;
    for (int s = 0; s < S; ++s) {
        const unsigned m = __ballot_sync(0xffffffffu, sp == s);
        if (m == 0) continue;
        int base = 0;
        if (lane == __ffs(m) - 1) base = atomicAdd(&sp_count[s], __popc(m));
        base = __shfl_sync(0xffffffffu, base, __ffs(m) - 1);
        if (sp == s) sp_rows[(size_t)s * n_total + base + __popc(m & ((1u << lane) - 1))] = a;
    }
}

__device__ __forceinline__ float celu_f(float x, float alpha, float inv_alpha)
{
    return x > 0.f ? x : alpha * (__expf(x * inv_alpha) - 1.0f);
}
// CELU'(z) expressed through h = CELU(z): 1 for h > 0, else exp(z/alpha) = h/alpha + 1
__device__ __forceinline__ float dcelu_from_h(float h, float inv_alpha)
{
    return h > 0.f ? 1.0f : fmaf(h, inv_alpha, 1.0f);
}

// v0: fp32 CUDA-core evaluation, TM rows per CTA, activations in shared memory.
template <int TM>
__global__ void __launch_bounds__(256)
k_mlp_f32(const MlpAll *__restrict__ M, int n_models, int L, int n_total, int n_atoms,
          const int *__restrict__ sp_rows, const int *__restrict__ sp_count, const float *__restrict__ aev,
          float *__restrict__ grad, double *__restrict__ energy, int *__restrict__ err)
{
    extern __shared__ __align__(16) float sm[];
    pdl_trigger();
    pdl_wait();               // the AEV rows (k_aev) are complete
    const int s = blockIdx.y;
    const int rows = sp_count[s];
    const int r0 = blockIdx.x * TM;
    if (r0 >= rows) return;
    __shared__ MlpDev N;      // network of (model blockIdx.z, species s)
    if (threadIdx.x < sizeof(MlpDev) / 4)
        reinterpret_cast<int *>(&N)[threadIdx.x] = reinterpret_cast<const int *>(&M->net[blockIdx.z][s])[threadIdx.x];
    __syncthreads();
    if (!N.loaded) { if (threadIdx.x == 0) atomicOr(err, kErrBitState); return; }
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int nrow = min(TM, rows - r0);
    const float alpha = N.alpha, inv_alpha = 1.0f / alpha;
    const float inv_m = 1.0f / (float)n_models;      // ensemble: mean of the energies and of dE/dAEV
    const int nl = N.n_layers;
    __shared__ int s_row[TM];
    if (tid < TM) s_row[tid] = tid < nrow ? sp_rows[(size_t)s * n_total + r0 + tid] : -1;
    __syncthreads();

    // activation buffers: h[0] = AEV rows, h[l] for hidden layers
    float *h[kMaxMlpLayers + 1];
    {
        float *p = sm;
        for (int l = 0; l < nl; ++l) { h[l] = p; p += TM * N.dims[l]; }
        h[nl] = p;
    }
    for (int t = tid; t < TM * (L / 4); t += 256) {
        const int r = t / (L / 4), c4 = t - r * (L / 4);
        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
        if (s_row[r] >= 0) v = reinterpret_cast<const float4 *>(aev + (size_t)s_row[r] * L)[c4];
        reinterpret_cast<float4 *>(h[0] + r * L)[c4] = v;
    }
    __syncthreads();

    // forward, hidden layers
    for (int l = 0; l < nl - 1; ++l) {
        const int K = N.dims[l], No = N.dims[l + 1];
        const float *W = N.w[l];
        for (int o = tid; o < No; o += 256) {
            float acc[TM];
            const float bb = N.b[l][o];
#pragma unroll
            for (int r = 0; r < TM; ++r) acc[r] = bb;
            for (int k = 0; k < K; k += 4) {
                const float w0 = W[(size_t)k * No + o], w1 = W[(size_t)(k + 1) * No + o];
                const float w2 = W[(size_t)(k + 2) * No + o], w3 = W[(size_t)(k + 3) * No + o];
#pragma unroll
                for (int r = 0; r < TM; ++r) {
                    const float4 x = *reinterpret_cast<const float4 *>(h[l] + r * K + k);
                    acc[r] = fmaf(x.x, w0, acc[r]); acc[r] = fmaf(x.y, w1, acc[r]);
                    acc[r] = fmaf(x.z, w2, acc[r]); acc[r] = fmaf(x.w, w3, acc[r]);
                }
            }
#pragma unroll
            for (int r = 0; r < TM; ++r) h[l + 1][r * No + o] = celu_f(acc[r], alpha, inv_alpha);
        }
        __syncthreads();
    }
    // last layer (one output): warp per row; energy summed in fp64
    {
        const int K = N.dims[nl - 1];
        const float *W = N.w[nl - 1];
        for (int r = wid; r < nrow; r += 8) {
            float acc = 0.f;
            for (int k = lane; k < K; k += 32) acc = fmaf(h[nl - 1][r * K + k], W[k], acc);
#pragma unroll
            for (int o = 16; o >= 1; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
            if (lane == 0) atomicAdd(&energy[s_row[r] / n_atoms], (double)(acc + N.b[nl - 1][0]) * (double)inv_m);
        }
    }
    __syncthreads();   // the backward chain below overwrites h[nl-1] in place
    // backward: d[nl-1][r][k] = W_last[k] * celu'(h[nl-1][r][k]), in place
    {
        const int K = N.dims[nl - 1];
        const float *W = N.w[nl - 1];
        for (int t = tid; t < TM * K; t += 256) {
            const int k = t % K;
            h[nl - 1][t] = W[k] * dcelu_from_h(h[nl - 1][t], inv_alpha);
        }
        __syncthreads();
    }
    for (int l = nl - 2; l >= 0; --l) {
        // d_in[r][k] = sum_o W^l[k][o] d_out[r][o]   (times celu'(h[l]) unless l == 0)
        const int K = N.dims[l], No = N.dims[l + 1];
        const float *WT = N.wt[l];       // [No][K]
        const float *dout = h[l + 1];
        for (int k = tid; k < K; k += 256) {
            float acc[TM];
#pragma unroll
            for (int r = 0; r < TM; ++r) acc[r] = 0.f;
            for (int o = 0; o < No; o += 4) {
                const float w0 = WT[(size_t)o * K + k], w1 = WT[(size_t)(o + 1) * K + k];
                const float w2 = WT[(size_t)(o + 2) * K + k], w3 = WT[(size_t)(o + 3) * K + k];
#pragma unroll
                for (int r = 0; r < TM; ++r) {
                    const float4 d = *reinterpret_cast<const float4 *>(dout + r * No + o);
                    acc[r] = fmaf(d.x, w0, acc[r]); acc[r] = fmaf(d.y, w1, acc[r]);
                    acc[r] = fmaf(d.z, w2, acc[r]); acc[r] = fmaf(d.w, w3, acc[r]);
                }
            }
            if (l > 0) {
#pragma unroll
                for (int r = 0; r < TM; ++r)
                    h[l][r * K + k] = acc[r] * dcelu_from_h(h[l][r * K + k], inv_alpha);
            } else {
#pragma unroll
                for (int r = 0; r < TM; ++r)
                    if (r < nrow) {
                        if (n_models == 1) grad[(size_t)s_row[r] * L + k] = acc[r];
                        else atomicAdd(&grad[(size_t)s_row[r] * L + k], acc[r] * inv_m);      // grad was zeroed
                    }
            }
        }
        __syncthreads();
    }
}

}  // namespace

namespace aevb {

void mlp_tc_pack(const float *w, int K_in, int N_out, std::vector<__nv_bfloat16> &fwd, std::vector<__nv_bfloat16> &bwd,
                 bool *exact);

static void free_net(MlpNet &n)
{
    for (int l = 0; l < kMaxMlpLayers; ++l) {
        cudaFree(n.w_fwd[l]); cudaFree(n.w_bwd[l]); cudaFree(n.w_f32[l]); cudaFree(n.w_t[l]); cudaFree(n.bias[l]);
    }
    memset(&n, 0, sizeof(n));
}

void mlp_free(aev_ctx *c)
{
    for (int m = 0; m < kMaxModels; ++m)
        for (int s = 0; s < kMaxS; ++s) free_net(c->nets[m][s]);
    cudaFree(c->f32_dev);
    c->f32_dev = nullptr;
}

int mlp_group(aev_ctx *c, const int32_t *species, int n_total, int batch, double *energy_out, cudaStream_t st)
{
    AEVB_CUDA(cudaMemsetAsync(c->sp_count, 0, (size_t)kMaxS * sizeof(int), st));
    k_group<<<(n_total + 255) / 256, 256, 0, st>>>(n_total, c->dp.S, species, c->sp_rows, c->sp_count, energy_out, batch);
    c->launches += 1;
    return cudaGetLastError() == cudaSuccess ? AEV_OK : AEV_ERR_CUDA;
}

// Device table of the fp32 kernel; rebuilt whenever a network is (re)loaded.  Syncs.
static int mlp_f32_upload(aev_ctx *c)
{
    // 8 KB, built on the heap per call: two contexts may load networks from two host threads at once
    std::unique_ptr<MlpAll> Mp(new MlpAll);
    MlpAll &M = *Mp;
    memset(&M, 0, sizeof(M));
    for (int m = 0; m < c->n_models; ++m)
        for (int s = 0; s < c->dp.S; ++s) {
            const MlpNet &n = c->nets[m][s];
            MlpDev &d = M.net[m][s];
            d.loaded = n.loaded; d.n_layers = n.n_layers; d.alpha = n.alpha;
            for (int l = 0; l <= n.n_layers; ++l) d.dims[l] = n.dims[l];
            for (int l = 0; l < n.n_layers; ++l) { d.w[l] = n.w_f32[l]; d.wt[l] = n.w_t[l]; d.b[l] = n.bias[l]; }
        }
    if (!c->f32_dev) AEVB_CUDA(cudaMalloc(&c->f32_dev, sizeof(MlpAll)));
    AEVB_CUDA(cudaMemcpy(c->f32_dev, &M, sizeof(MlpAll), cudaMemcpyHostToDevice));
    return AEV_OK;
}

int mlp_forward_backward(aev_ctx *c, const int32_t *species, int n_total, int n_atoms, int batch,
                         const float *aev, float *grad_aev, double *energy_out, cudaStream_t st)
{
    const int S = c->dp.S, L = c->dp.L, nm = c->n_models;
    int sum_hidden = 0;
    bool all_tc = true;
    for (int m = 0; m < nm; ++m)
        for (int s = 0; s < S; ++s) {
            const MlpNet &n = c->nets[m][s];
            if (!n.loaded) continue;
            int sh = 0;
            for (int l = 0; l < n.n_layers; ++l) sh += n.dims[l];
            if (sh > sum_hidden) sum_hidden = sh;
            if (!n.tc_ok) all_tc = false;
        }
    prof_begin(c, 5, st);
    // tensor-core path when every loaded network qualifies (ani_mlp_tc.cu); else fp32 CUDA cores
    if (all_tc && !(c->hp.flags & AEV_FLAG_MLP_FP32)) {
        const int rc = mlp_tc_forward_backward(c, n_total, n_atoms, aev, grad_aev, energy_out, st);
        prof_end(c, st);
        c->launches += 1;
        return rc;
    }
    constexpr int TM = 8;
    const size_t smem = (size_t)TM * sum_hidden * sizeof(float);
    if (smem > 200 * 1024) return AEV_ERR_UNSUPPORTED;
    if (smem > c->mlp_smem_optin) {
        AEVB_CUDA(cudaFuncSetAttribute(k_mlp_f32<TM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        c->mlp_smem_optin = smem;
    }
    if (!c->f32_dev) return AEV_ERR_STATE;
    dim3 grid((n_total + TM - 1) / TM, S, nm);
    if ((c->hp.flags & AEV_FLAG_DETERMINISTIC) && nm > 1) {      // one launch per model: the models' adds arrive in model order
        grid.z = 1;
        for (int m = 0; m < nm; ++m) {
            const MlpAll *row = reinterpret_cast<const MlpAll *>(static_cast<const MlpAll *>(c->f32_dev)->net + m);
            launch_pdl(k_mlp_f32<TM>, grid, dim3(256), smem, st, row, nm, L, n_total, n_atoms,
                       (const int *)c->sp_rows, (const int *)c->sp_count, aev, grad_aev, energy_out, c->ws.err);
        }
        c->launches += nm - 1;
    } else
    launch_pdl(k_mlp_f32<TM>, grid, dim3(256), smem, st, static_cast<const MlpAll *>(c->f32_dev), nm, L, n_total, n_atoms,
               (const int *)c->sp_rows, (const int *)c->sp_count, aev, grad_aev, energy_out, c->ws.err);
    prof_end(c, st);
    c->launches += 1;
    if (cudaGetLastError() != cudaSuccess) return AEV_ERR_CUDA;
    return AEV_OK;
}

}  // namespace aevb

extern "C" int ani_mlp_kernel(const aev_ctx *c)
{
    if (!c) return AEV_ERR_INVALID_ARG;
    bool any = false, all_tc = true;
    for (int m = 0; m < c->n_models; ++m)
        for (int s = 0; s < c->dp.S; ++s) {
            const MlpNet &n = c->nets[m][s];
            if (!n.loaded) continue;
            any = true;
            if (!n.tc_ok) all_tc = false;
        }
    if (!any) return AEV_ERR_STATE;
    return (all_tc && !(c->hp.flags & AEV_FLAG_MLP_FP32)) ? 1 : 0;
}

extern "C" int ani_mlp_set_ensemble(aev_ctx *c, int32_t n_models)
{
    if (!c || n_models < 1 || n_models > kMaxModels) return AEV_ERR_INVALID_ARG;
    DeviceGuard guard(c->device);
    if (!guard.ok()) return AEV_ERR_CUDA;
    AEVB_CUDA(cudaDeviceSynchronize());
    for (int m = 0; m < kMaxModels; ++m)
        for (int s = 0; s < kMaxS; ++s) free_net(c->nets[m][s]);
    c->n_models = n_models;
    if (c->hg_exec) { cudaGraphExecDestroy(c->hg_exec); c->hg_exec = nullptr; }
    c->hg_state = 0;      // a captured host-call graph has the old networks baked in
    return AEV_OK;
}

extern "C" int ani_mlp_load_model(aev_ctx *c, int32_t model, int32_t species, int32_t n_layers, const int32_t *dims,
                                  const float *const *weights, const float *const *biases, float celu_alpha)
{
    if (!c || !dims || !weights || !biases) return AEV_ERR_INVALID_ARG;
    if (species < 0 || species >= c->dp.S || model < 0 || model >= c->n_models) return AEV_ERR_INVALID_ARG;
    if (n_layers < 2 || n_layers > kMaxMlpLayers) return AEV_ERR_UNSUPPORTED;
    if (dims[0] != c->dp.L || dims[n_layers] != 1) return AEV_ERR_INVALID_ARG;
    if (!(celu_alpha > 0.f)) return AEV_ERR_INVALID_ARG;
    for (int l = 1; l < n_layers; ++l)
        if (dims[l] < 16 || dims[l] > 256 || dims[l] % 16) return AEV_ERR_UNSUPPORTED;
    for (int l = 0; l < n_layers; ++l)
        if (!weights[l] || !biases[l]) return AEV_ERR_INVALID_ARG;
    // all models of one species share one shape (one launch geometry per species)
    for (int m = 0; m < c->n_models; ++m) {
        const MlpNet &o = c->nets[m][species];
        if (m == model || !o.loaded) continue;
        if (o.n_layers != n_layers) return AEV_ERR_INVALID_ARG;
        for (int l = 0; l <= n_layers; ++l)
            if (o.dims[l] != dims[l]) return AEV_ERR_INVALID_ARG;
    }
    DeviceGuard guard(c->device);
    if (!guard.ok()) return AEV_ERR_CUDA;
    AEVB_CUDA(cudaDeviceSynchronize());
    if (c->hg_exec) { cudaGraphExecDestroy(c->hg_exec); c->hg_exec = nullptr; }
    c->hg_state = 0;      // a captured host-call graph has the old networks baked in
    MlpNet &n = c->nets[model][species];
    free_net(n);
    n.n_layers = n_layers;
    n.bf16_exact = 1;
    n.alpha = celu_alpha;
    for (int l = 0; l <= n_layers; ++l) n.dims[l] = dims[l];
    for (int l = 0; l < n_layers; ++l) {
        const int K = dims[l], No = dims[l + 1];
        const size_t cnt = (size_t)K * No;
        std::vector<float> wt(cnt);
        std::vector<__nv_bfloat16> fw, bw;
        bool exact = true;
        mlp_tc_pack(weights[l], K, No, fw, bw, &exact);
        if (l < n_layers - 1 && !exact) n.bf16_exact = 0;
        for (int k = 0; k < K; ++k)
            for (int o = 0; o < No; ++o) wt[(size_t)o * K + k] = weights[l][(size_t)k * No + o];
        AEVB_CUDA(cudaMalloc((void **)&n.w_f32[l], cnt * 4));
        AEVB_CUDA(cudaMalloc((void **)&n.w_t[l], cnt * 4));
        AEVB_CUDA(cudaMalloc(&n.w_fwd[l], fw.size() * 2));
        AEVB_CUDA(cudaMalloc(&n.w_bwd[l], bw.size() * 2));
        AEVB_CUDA(cudaMalloc((void **)&n.bias[l], (size_t)No * 4));
        AEVB_CUDA(cudaMemcpy(n.w_f32[l], weights[l], cnt * 4, cudaMemcpyHostToDevice));
        AEVB_CUDA(cudaMemcpy(n.w_t[l], wt.data(), cnt * 4, cudaMemcpyHostToDevice));
        AEVB_CUDA(cudaMemcpy(n.w_fwd[l], fw.data(), fw.size() * 2, cudaMemcpyHostToDevice));
        AEVB_CUDA(cudaMemcpy(n.w_bwd[l], bw.data(), bw.size() * 2, cudaMemcpyHostToDevice));
        AEVB_CUDA(cudaMemcpy(n.bias[l], biases[l], (size_t)No * 4, cudaMemcpyHostToDevice));
    }
    n.b_last = biases[n_layers - 1][0];
    n.tc_ok = mlp_tc_eligible(n, c->dp.L) ? 1 : 0;
    n.loaded = 1;
    int rc = mlp_f32_upload(c);
    if (rc) return rc;
    return mlp_tc_upload(c);
}

extern "C" int ani_mlp_load(aev_ctx *c, int32_t species, int32_t n_layers, const int32_t *dims,
                            const float *const *weights, const float *const *biases, float celu_alpha)
{
    return ani_mlp_load_model(c, 0, species, n_layers, dims, weights, biases, celu_alpha);
}

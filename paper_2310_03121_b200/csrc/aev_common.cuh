// aev_common.cuh -- context, device-side parameter block and small helpers shared by the
// translation units of libaev_b200.so (aev_kernels.cu, ani_mlp.cu).  Product code: shares
// nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include "../../include/aev.h"

namespace aevb {

constexpr int kNR = 16;        // radial shifts   (BASELINE.json:configs[0])
constexpr int kNA = 4;         // angular radial shifts  (the ANI-1x-style default; 8 x 4 is the other supported split)
constexpr int kNZ = 8;         // angular angle shifts
constexpr int kBlk = kNA * kNZ;  // 32 entries per species-pair block, whatever the split
constexpr int kMaxNA = 8, kMaxNZ = 8;
constexpr int kMaxS = 8;
constexpr int kSpeciesShift = 26;  // neighbour entry .w = caller index of j | species << 26
constexpr int kIdxMask = (1 << kSpeciesShift) - 1;
constexpr int kMaxMlpLayers = 4;
constexpr int kMaxModels = 8;      // networks per species in an ensemble

// Everything the kernels need about the symmetry functions; passed by value (constant bank).
struct DevParams {
    int S, L, rad_len, n_blocks, zeta_log2;
    int n_a;                     // angular radial shifts: 4 (x 8 angle shifts) or 8 (x 4)
    float rcr, rca, rcr2, rca2;
    float eta_r, eta_a;          // natural units (for derivatives)
    float eta_r_l2, eta_a_l2;    // eta * log2(e)    (for ex2)
    float inv_rcr, inv_rca;      // 1/R  (cutoff function argument r/R, used with cospi/sinpi)
    float zeta_half;             // zeta / 2
    float c, c2, one_m_c2;       // cos_scale, its square, 1 - c^2
    float shf_r[kNR];
    float shf_a[kMaxNA];
    float cz[kMaxNZ], sz[kMaxNZ];      // cos / sin of the angle shifts
    unsigned long long half2, neta_r2;                 // (0.5, 0.5) and (-eta_r log2 e) twice
    unsigned long long nshf_r2[kNR / 2];               // -shf_r, packed pairs (m even | m odd << 32)
    unsigned long long hcz2[kMaxNZ / 2], hsz2[kMaxNZ / 2];   // cos/2, sin/2 of the angle shifts, packed pairs (z even | z odd << 32)
};

// Geometry of one call (filled on the host per call, passed by value).
struct Geom {
    int n_atoms, batch, n_total;
    int periodic;                // 1: cell grid with a 27-cell stencil and image shifts per stencil cell
    int mi;                      // 1: one cell per system, all pairs, minimum image taken in the distance test (boxes
                                 //    with fewer than 3 cells along an edge, and every triclinic box)
    float lat[9];                // mi: lattice rows a = (ax,0,0), b = (bx,by,0), c = (cx,cy,cz) (orthorhombic: diagonal)
    float inv_diag[3];           // mi: 1/ax, 1/by, 1/cz
    int ncx, ncy, ncz, ncell;    // cells per system (non-periodic: 1,1,1,1)
    int nbins;                   // batch*ncell*S
    int bin_cap;                 // capacity of one (cell,species) member list
    int cap_r, cap_a;            // per-atom neighbour capacities (total radial / angular)
    int cand_cap;                // shared-memory candidate tile capacity (float4 entries)
    float box[3], inv_box[3], cell_scale[3];   // cell_scale = nc / L
    int c_first, c_count;        // central atoms k_aev / k_backward evaluate: flat indices [c_first, c_first + c_count)
                                 // (all of them unless aev_forward_range asked for a slab)
};

// Device workspace owned by the context.
struct Workspace {
    int *bin_cnt;        // [nbins_cap] member counts (zero between calls: cleared by k_nbr)
    float4 *cpos;        // [nbins_cap*bin_cap] bin members: wrapped position, caller index | species << 26
    float4 *cpos_sorted; // the same ordered by caller index inside every bin (AEV_FLAG_DETERMINISTIC, k_rank)
    int *abin;           // [n_total] bin of every atom (AEV_FLAG_DETERMINISTIC)
    float4 *nlist;       // [n_total][cap_r] neighbour entries (dx,dy,dz, caller index j | s<<26), angular first
    int2 *ncount;        // [n_total] (nA, nB)
    int4 *hdr;           // [n_total] per atom (caller order): (nA, nB, caller index, species)
    int *noff;           // [n_total][kMaxS+1] per-species list offsets: offA | offB << 16
    int *err;            // device error flags (bitmask)
    // Verlet-skin reuse (aev_params.skin > 0): lists built with rcr+skin / rca+skin, filtered every call by k_refresh
    float4 *vlist;       // [n_total][vcap_r]
    int2 *vcount;        // [n_total]
    int4 *vhdr;          // [n_total]
    int *vnoff;          // [n_total][kMaxS+1]
    float *pos_ref;      // [n_total][3] positions at the last build
    float4 *pos4;        // [n_total] this call's positions, padded (k_disp writes, k_refresh gathers)
    int *need;           // 1: this call rebuilds the Verlet lists (set by k_disp, cleared by k_refresh); NULL without skin
    int *valid;          // 1: the Verlet lists match the current shapes (set by k_nbr, cleared by the host)
    unsigned long long *builds;   // Verlet-list builds so far
    float4 *f4acc;       // [n_total] padded fp32 force accumulator (default mode), zero between calls
    long long *facc;     // [n_total][3] fixed-point force accumulator (AEV_FLAG_DETERMINISTIC), zero between calls
    unsigned *nbr_done;  // k_nbr CTAs that have read their bin counters (reset by the last one)
    unsigned long long *pair_count;  // export counter
};

struct MlpNet {
    int loaded;
    int n_layers;
    int dims[kMaxMlpLayers + 1];
    // tensor-core operands (ani_mlp_tc.cu): bf16 hi part | bf16 residual part of every weight, chunked K-major
    void *w_fwd[kMaxMlpLayers];  // forward operand  hi [in/8][out][8] | lo (same shape)
    void *w_bwd[kMaxMlpLayers];  // backward operand hi [out/8][in][8] | lo
    int bf16_exact;              // every hidden-layer weight is bf16-representable (the lo operands are all zero)
    int tc_ok;                   // shape qualifies for the tcgen05 kernel
    float alpha;                 // CELU alpha of this network
    float b_last;                // bias of the last (N = 1) layer
    float *w_f32[kMaxMlpLayers]; // f32 [in][out] as given
    float *w_t[kMaxMlpLayers];   // f32 [out][in] (transposed copy for the backward chain)
    float *bias[kMaxMlpLayers];  // f32 [out]
};

}  // namespace aevb

struct aev_ctx {
    aev_params hp;               // host copy of the parameters (pointers nulled)
    aevb::DevParams dp;
    aevb::Geom geom;             // geometry of the most recent neighbour build
    aevb::Workspace ws;
    int device;
    int sm_count;
    int state;                   // 0 none, 1 neighbours built, 2 forward done
    int64_t launches;
    cudaStream_t last_stream;
    size_t cap_total;            // atoms the workspace is sized for
    size_t nbins_cap, members_cap;
    int vcap_r, vcap_a;          // per-atom capacities of the Verlet lists
    aevb::Geom vgeom;            // geometry of the last call in skin mode (a change invalidates the Verlet lists)
    int vgeom_set;
    int next_first, next_count;  // central-atom range of the NEXT launch_neighbors (aev_forward_range); count < 0 = all
    int fwd_smem_optin;          // bytes of dynamic smem the forward kernels were opted into (per device => per ctx)
    size_t bwd_smem_optin, mlp_smem_optin;
    int tc_smem_optin;
    // MLP
    aevb::MlpNet nets[aevb::kMaxModels][aevb::kMaxS];
    int n_models;                // ensemble size (1 unless ani_mlp_set_ensemble was called)
    size_t mlp_cap;              // atoms the MLP workspaces are sized for
    float *mlp_aev;              // [n_total][L]   (ani_energy_forces workspace)
    float *mlp_grad;             // [n_total][L]
    void *mlp_work;              // MLP scratch (activations)
    size_t mlp_work_bytes;
    int *sp_rows;                // [S][n_total] caller indices grouped by species
    int *sp_count;               // [S]
    void *tc_dev;                // device copy of the tensor-core network table (ani_mlp_tc.cu)
    void *f32_dev;               // device copy of the fp32 network table (ani_mlp.cu)
    float *sub_buf;              // [max_atoms][3] gathered positions | [max_atoms][3] forces (ani_energy_forces_subset)
    // host staging (pinned) + device staging for the *_host entry points
    int profiling;
    void *prof;                  // std::vector<ProfRec>* (aev_kernels.cu)
    void *h_pin; size_t h_pin_bytes;
    void *d_stage; size_t d_stage_bytes;
    cudaStream_t s_main, s_h2d, s_d2h;      // streams of the host entry points (kernels, big H2D, big D2H)
    cudaEvent_t ev_fwd, ev_grad;
    // ani_energy_forces_host: the whole evaluation (H2D, kernels, D2H) as a CUDA graph, captured on the second call
    // with the same shapes and box and replayed from then on (an MD engine calls it every step: 13 enqueue calls -> 1)
    cudaGraphExec_t hg_exec;
    int hg_state;                // 0: nothing seen, 1: one eager call with this key seen, 2: graph ready, -1: capture failed
    int hg_n, hg_batch, hg_boxn;
    float hg_box[9];
    int64_t hg_launches;         // kernels per replay
    aevb::Geom hg_geom, hg_vgeom; // c->geom / c->vgeom as the captured evaluation left them (restored after every replay)
};

namespace aevb {

#define AEVB_CUDA(call)                                   \
    do {                                                  \
        cudaError_t e__ = (call);                         \
        if (e__ != cudaSuccess) return AEV_ERR_CUDA;      \
    } while (0)

enum { kErrBitCapacity = 1, kErrBitState = 2, kErrBitCheck = 4 };

// -DAEVB_CHECKS (debug builds; compute-sanitizer is not available on every pool): bounds checks of the computed list
// slots and shared-memory indices; a failed check raises kErrBitCheck, which aev_status reports as AEV_ERR_CUDA.
#ifdef AEVB_CHECKS
#define AEVB_CHECK(errp, cond) do { if (!(cond)) atomicOr((errp), kErrBitCheck); } while (0)
#else
#define AEVB_CHECK(errp, cond) do { } while (0)
#endif

// Every entry point runs on the context's device and leaves the caller's current device as it found it.
class DeviceGuard {
public:
    explicit DeviceGuard(int dev) : prev_(-1), ok_(false)
    {
        if (cudaGetDevice(&prev_) != cudaSuccess) { prev_ = -1; return; }
        ok_ = (prev_ == dev) || cudaSetDevice(dev) == cudaSuccess;
        if (prev_ == dev) prev_ = -1;      // nothing to restore
    }
    ~DeviceGuard() { if (prev_ >= 0) cudaSetDevice(prev_); }
    bool ok() const { return ok_; }
private:
    int prev_;
    bool ok_;
};

// Programmatic dependent launch: a kernel launched with launch_pdl() may become resident while its
// predecessor in the stream is still draining; it must pass pdl_wait() before it touches anything the
// predecessor (or, transitively, an earlier kernel) wrote.  pdl_trigger() lets the successor start early.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args)
{
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// species partition for the MLP (ani_mlp.cu): memset of the counters + k_group
int mlp_group(aev_ctx *c, const int32_t *species, int n_total, int batch, double *energy_out, cudaStream_t st);

// MLP entry points implemented in ani_mlp.cu
int mlp_forward_backward(aev_ctx *c, const int32_t *species, int n_total, int n_atoms, int batch,
                         const float *aev, float *grad_aev, double *energy_out,
                         cudaStream_t st);
void mlp_free(aev_ctx *c);
// tcgen05 path (ani_mlp_tc.cu)
bool mlp_tc_eligible(const MlpNet &n, int L);
int mlp_tc_upload(aev_ctx *c);
int mlp_tc_forward_backward(aev_ctx *c, int n_total, int n_atoms, const float *aev, float *grad_aev,
                            double *energy_out, cudaStream_t st);
// profiling brackets (aev_kernels.cu): slot 0 bin (k_bin, k_rank), 1 fout (k_fout / k_fixout), 2 aev (k_aev), 3 backward,
// 4 nbr (k_nbr, k_refresh), 5 mlp
void prof_begin(aev_ctx *c, int slot, cudaStream_t st);
void prof_end(aev_ctx *c, cudaStream_t st);

}  // namespace aevb

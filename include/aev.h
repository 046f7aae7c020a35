/*
 * aev.h -- C ABI of libaev_b200.so: the B200-native (sm_100a) hot path of an ANI-style
 * ML-potential force evaluation inside an MD step.
 *
 * What the path is for: "a model that takes atomic positions as input and computes
 * potential energy.  Forces can be automatically calculated through backpropagation, or
 * ... returned explicitly" (section "OpenMM-Torch").  Which operations it
 * consists of: "computing the atom-centered symmetry functions used in the ANI family of
 * potentials, building neighbor lists" (section "Optimization Through
 * NNPOps").  The paper prints no formulas; the formulas are BASELINE.json:north_star's
 * steps (1)-(4) as restated in SURVEY.md section 8(c) and DESIGN.md section 3:
 *
 *   (1) pairs    d_ij = x_j - x_i - L*rint((x_j - x_i)/L)  (orthorhombic minimum image),
 *                radial set r_ij < rcr, angular set r_ij < rca   (strict <)
 *   (2) radial   G_R[i][s*nR+m]  = sum_{j in radial set, s_j=s}
 *                                  0.25*exp(-eta_r*(r_ij-shf_r[m])^2)*fc(r_ij; rcr)
 *   (3) angular  G_A[i][S*nR + p(s_j,s_k)*nA*nZ + a*nZ + z] = sum over UNORDERED {j,k} in
 *                the angular set of
 *                2^(1-zeta)*(1+cos(theta-shf_z[z]))^zeta*exp(-eta_a*((r_ij+r_ik)/2-shf_a[a])^2)
 *                *fc(r_ij; rca)*fc(r_ik; rca),   theta = acos(cos_scale * cos(angle j-i-k)),
 *                p(s1<=s2) = s1*(2S-s1-1)/2 + s2,   fc(r;R) = 0.5*cos(pi*r/R)+0.5
 *   (4) backward forces[a] = - sum_i sum_slot grad_aev[i][slot] * dAEV[i][slot]/dx_a,
 *                then per-species MLPs  z = hW+b, CELU_alpha hidden, linear last layer,
 *                E = sum_i NN_{s_i}(AEV_i)                     (BASELINE.json:configs[4])
 *
 * Conventions for every call
 *   - plain pointers and sizes only; "device" pointers are CUDA device pointers on the
 *     context's device, "host" pointers are ordinary host memory;
 *   - the caller owns every buffer passed in; the library never frees them and keeps no
 *     pointer to them after the call returns (it copies what aev_backward needs into
 *     workspace owned by the context);
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream);
 *     device-pointer calls are asynchronous on that stream unless marked "syncs";
 *   - every call returns 0 (AEV_OK) or a negative AEV_ERR_* code; nothing throws, prints
 *     or exits;
 *   - a context is used from one host thread and one stream at a time;
 *   - there is no CPU fallback and no other backend: a device that is not compute
 *     capability 10.x gives AEV_ERR_UNSUPPORTED.
 *
 * Supported parameter space (else AEV_ERR_UNSUPPORTED): 1 <= num_species <= 8,
 * n_shf_r == 16, (n_shf_a, n_shf_z) == (4, 8) - the shift counts of BASELINE.json:configs[0],
 * "ANI-1x-style" - or (8, 4) (the lane mappings of the kernels are built on 16 and on 32 = 4 x 8 = 8 x 4), 1 <= zeta <= 64
 * (powers of two by repeated squaring, any other value - e.g. 14.1 - as exp2(zeta log2 b) on the SFU), 0 < rca <= rcr, 0 < cos_scale <= 1; periodic boxes are orthorhombic (three
 * edge lengths, each >= 2*rcr) or, with AEV_FLAG_TRICLINIC, reduced triclinic (three lattice
 * vectors, ax, by, cz >= 2*rcr).  Orthorhombic boxes with at least 3 cells of edge >= rcr along every
 * axis use the cell list; smaller ones and every triclinic box are searched as one cell with the
 * minimum image taken per pair (O(n^2) candidate tests: meant for ML regions of a few hundred atoms,
 * such as the 528-atom periodic cell of PAPER.md:223).
 */
#ifndef AEV_B200_H
#define AEV_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    AEV_OK = 0,
    AEV_ERR_INVALID_ARG = -1,   /* null pointer, bad shape, n > max_atoms, ...                 */
    AEV_ERR_BOX_TOO_SMALL = -2, /* a periodic edge (triclinic: ax, by or cz) < 2*rcr: no unique minimum image  */
    AEV_ERR_CAPACITY = -3,      /* a per-atom neighbour capacity or a cell capacity overflowed
                                   on the device; results of that call are incomplete          */
    AEV_ERR_STATE = -4,         /* aev_backward without a preceding aev_forward, MLP not loaded */
    AEV_ERR_UNSUPPORTED = -5,   /* parameter combination or device outside the supported space  */
    AEV_ERR_CUDA = -6,          /* a CUDA runtime call failed                                   */
    AEV_ERR_STATIC_LIMIT = -7   /* aev_pairs_static: more atoms than its fixed, statically allocated working
                                   memory holds (AEV_STATIC_MAX_ATOMS); use a context instead    */
};

typedef struct aev_ctx aev_ctx; /* opaque; owns all device workspace */

/* aev_params.flags */
enum {
    AEV_FLAG_DETERMINISTIC = 1, /* bit-identical AEV and forces run to run: the members of
                                   every cell are ordered by atom index before the neighbour search (by default they
                                   keep the order the binning atomics ran in, so AEV sums agree to rounding only),
                                   and aev_backward accumulates the contributions on neighbours in 64-bit fixed point
                                   (2^-32 force units) instead of fp32 REDs; with an ensemble the networks run as one
                                   launch per model, so the mean dE/dAEV - and the forces of ani_energy_forces - are
                                   summed in model order.  Energies are fp64 atomic sums and agree to fp64 rounding
                                   only.  A little slower.                                                          */
    AEV_FLAG_MLP_FP32 = 2,      /* debugging: run the fp32 CUDA-core MLP kernel even where the tcgen05
                                   kernel qualifies                                                     */
    AEV_FLAG_TRICLINIC = 4      /* every `box` argument is HOST f32[9]: lattice vectors a, b, c as rows,
                                   in reduced form a = (ax,0,0), b = (bx,by,0), c = (cx,cy,cz) with
                                   ax, by, cz > 0, |bx| <= ax/2, |cx| <= ax/2, |cy| <= by/2             */
};

typedef struct {
    int32_t num_species;        /* S; species ids are 0..S-1, id < 0 marks a padding atom       */
    float rcr, rca;             /* radial / angular cutoff, same length unit as positions       */
    float eta_r;
    int32_t n_shf_r;
    const float *shf_r;         /* HOST pointer, n_shf_r values, copied at create               */
    float eta_a, zeta;
    int32_t n_shf_a;
    const float *shf_a;         /* HOST, n_shf_a values                                         */
    int32_t n_shf_z;
    const float *shf_z;         /* HOST, n_shf_z values (radians)                               */
    float cos_scale;            /* 1.0 = the literal north_star formula; 0.95 = damped variant  */
    int32_t max_atoms;          /* capacity: atoms per system                                   */
    int32_t max_batch;          /* capacity: systems per call                                   */
    int32_t max_radial_nbrs;    /* per-atom capacity for r < rcr (0 = default 128)              */
    int32_t max_angular_nbrs;   /* per-atom capacity for r < rca (0 = default 48; <= 64)        */
    int32_t device;             /* CUDA ordinal                                                 */
    uint32_t flags;             /* AEV_FLAG_* bits, 0 = defaults                                */
    float skin;                 /* Verlet skin (same length unit). 0 = the neighbour structure is
                                   rebuilt in every aev_forward (reading G18, the headline protocol).
                                   > 0: lists are built with cutoffs rcr+skin / rca+skin and reused by
                                   later calls with the same shapes until some atom has moved more than
                                   skin/2 since the build (checked on the device, CUDA-graph safe); the
                                   exact cutoffs are applied when the lists are read, so results do
                                   not depend on when the last rebuild happened (to rounding order).   */
} aev_params;

/* Creates a context (allocates workspace for max_batch*max_atoms atoms on `device`). Syncs. */
int aev_create(const aev_params *p, aev_ctx **out);
/* Frees the context and everything it owns. Syncs. NULL is accepted. */
int aev_destroy(aev_ctx *c);
/* L = S*n_shf_r + S*(S+1)/2*n_shf_a*n_shf_z (384 for S = 4). Negative on a NULL context. */
int aev_length(const aev_ctx *c);

/*
 * Step (1) only: cutoff neighbour search.
 *   pos      device f32 [batch][n_atoms][3]
 *   species  device i32 [batch][n_atoms]; id < 0 = padding atom (belongs to no pair)
 *   box      HOST f32[3] orthorhombic edge lengths (shared by the batch), or NULL =
 *            non-periodic all-pairs within each system.  Positions may lie outside [0,L).
 *            On a context created with AEV_FLAG_TRICLINIC: HOST f32[9], lattice rows a, b, c.
 * Builds, inside the context, per-atom neighbour lists (angular-set neighbours first) that
 * aev_export_pairs can read back.  Asynchronous.
 */
int aev_neighbors(aev_ctx *c, const float *pos, const int32_t *species, const float *box,
                  int32_t n_atoms, int32_t batch, void *stream);

/*
 * Steps (1)-(3): neighbour search (rebuilt in every call, reading G18, unless the context has a
 * Verlet skin - see aev_params.skin) + radial and angular AEV (rows A1-A4).
 *   aev_out  device f32 [batch][n_atoms][L], OVERWRITTEN, rows in the caller's atom order;
 *            rows of padding atoms are written as zeros.
 * Keeps what aev_backward needs inside the context.  Asynchronous.
 */
int aev_forward(aev_ctx *c, const float *pos, const int32_t *species, const float *box,
                int32_t n_atoms, int32_t batch, float *aev_out, void *stream);

/*
 * Step (4), first half (rows A5-A7), for the most recent aev_forward on this context:
 *   grad_aev    device f32 [batch][n_atoms][L]  upstream dE/dAEV
 *   forces_out  device f32 [batch][n_atoms][3], OVERWRITTEN,
 *               forces_out[a] = - sum_i sum_slot grad_aev[i][slot]*dAEV[i][slot]/dx_a
 * The centre's own terms are reduced with warp shuffles; the reaction on each radial
 * neighbour and the gradient on each angular neighbour are added with one 16-byte vector RED
 * into a padded accumulator of the context (copied to forces_out and cleared by a last small
 * kernel), so by default forces are reproducible to rounding, not bit for bit; with
 * AEV_FLAG_DETERMINISTIC they are accumulated in 64-bit fixed point and are bit-identical
 * run to run (so is the AEV then: every cell is searched in atom-index order, whether its
 * stencil fits the shared-memory stage or is scanned from global memory).
 * AEV_ERR_STATE if no forward precedes it.  Asynchronous.
 */
int aev_backward(aev_ctx *c, const float *grad_aev, float *forces_out, void *stream);

/*
 * A slab of the central atoms (sharding the evaluation over GPUs; the paper's only
 * parallelism content is multi-GPU MD over NVLink).  aev_forward_range is aev_forward for
 * the central atoms with flat index (b*n_atoms + a) in [first, first + count) only: the neighbour search still
 * covers every atom (a slab's neighbours lie outside it), but only the AEV rows of the slab are computed and
 * written - every other row of aev_out is left untouched.  The aev_backward that follows then reads grad_aev
 * rows [first, first + count) only and returns the PARTIAL forces
 *     forces_out[a] = - sum_{i in slab} sum_slot grad_aev[i][slot] * dAEV[i][slot]/dx_a      for ALL atoms a,
 * so the partial forces of disjoint slabs that cover the system add up to aev_backward's forces (to fp32 rounding).
 * One process per GPU evaluates its slab on the full position array and the partial forces are summed across ranks
 * (paper_2310_03121_b200/sharded.py: all-reduce over NCCL).  AEV_ERR_INVALID_ARG if the range is empty or leaves
 * [0, batch*n_atoms).  The range applies to this call and its aev_backward only.  Asynchronous.
 */
int aev_forward_range(aev_ctx *c, const float *pos, const int32_t *species, const float *box,
                      int32_t n_atoms, int32_t batch, int32_t first, int32_t count, float *aev_out,
                      void *stream);

/*
 * Loads the network of one species (rows A8-A9; BASELINE.json:configs[4]).
 *   dims     HOST i32 [n_layers+1]; dims[0] must equal L, dims[n_layers] must be 1,
 *            2 <= n_layers <= 4, hidden widths multiples of 16 and <= 256
 *   weights  HOST array of n_layers HOST pointers, layer l is f32 [dims[l]][dims[l+1]]
 *            row-major ("[in][out]")
 *   biases   HOST array of n_layers HOST pointers, f32 [dims[l+1]]
 * Hidden activations are CELU(alpha); the last layer is linear.  Syncs.
 * Which kernel runs (ani_mlp_kernel tells): the tcgen05 kernel takes a network with 1-3 hidden layers of width
 * 16..160 whose pre-activations fit the 512 TMEM columns (the hidden widths sum to <= 512, and for every hidden
 * layer l but the last, width_1 + .. + width_l + width_l <= 512: its backward accumulator sits behind z_1..z_l) and
 * whose inner-layer weight operands each fit one 48 KB shared-memory buffer, forward and transposed: for consecutive
 * hidden widths (a, b), ceil(a/64)*b <= 384 and ceil(b/64)*a <= 384 - so 128 -> 160 and 160 -> 128 qualify,
 * 144 -> 160 and 160 -> 160 do not.  Activations AND weights go in as bf16 hi + lo operands (hi*hi + lo*hi + hi*lo,
 * fp32 accumulate; the weight-lo MMA is skipped for a network whose weights are all bf16-representable).  Any other
 * shape, or any loaded network outside the envelope, makes the whole evaluation run the fp32 CUDA-core kernel.
 * ani_mlp_load == ani_mlp_load_model with model = 0 of an ensemble of 1.
 */
int ani_mlp_load(aev_ctx *c, int32_t species, int32_t n_layers, const int32_t *dims,
                 const float *const *weights, const float *const *biases, float celu_alpha);

/*
 * Ensemble of networks over one AEV ("ANI-2x ... is an ensemble of eight models").
 * ani_mlp_set_ensemble declares n_models (1..8) and drops every loaded network;
 * ani_mlp_load_model loads the network of (model, species); all models of one species must have
 * the same dims.  With an ensemble, ani_energy_forces returns the MEAN over the models of the
 * energy and of dE/dAEV (one AEV forward, one AEV backward).  Sync.
 */
int ani_mlp_set_ensemble(aev_ctx *c, int32_t n_models);
/* Which kernel ani_energy_forces runs for the networks loaded so far: 1 = tcgen05 tensor-core kernel,
 * 0 = fp32 CUDA-core kernel (a shape outside the envelope above, or AEV_FLAG_MLP_FP32),
 * AEV_ERR_STATE = no network loaded. */
int ani_mlp_kernel(const aev_ctx *c);
int ani_mlp_load_model(aev_ctx *c, int32_t model, int32_t species, int32_t n_layers,
                       const int32_t *dims, const float *const *weights,
                       const float *const *biases, float celu_alpha);

/*
 * The whole path: neighbours + AEV + per-species MLP forward/backward + AEV backward.
 *   energy_out  device f64 [batch]             E_b = sum_i NN_{s_i}(AEV_i)
 *   forces_out  device f32 [batch][n_atoms][3]  -dE/dx
 * Every species present must have a network loaded (else the device flag reports
 * AEV_ERR_STATE through aev_status).  Asynchronous.
 */
int ani_energy_forces(aev_ctx *c, const float *pos, const int32_t *species, const float *box,
                      int32_t n_atoms, int32_t batch, double *energy_out, float *forces_out,
                      void *stream);

/*
 * The ML region of a mixed ML/MM system (createMixedSystem(topology, mm_system, ml_atoms);
 * 53 ML atoms of 134,099): energy and forces of the n_ml atoms listed in ml_index, evaluated
 * as one non-batched system of their own (positions gathered from the full array by a kernel), and the
 * ML forces ADDED onto forces_all at those atoms (the MM forces already there are kept; every other
 * entry is left untouched).
 *   pos_all     device f32 [n_all][3]     positions of the whole system
 *   ml_index    device i32 [n_ml]         distinct indices into pos_all / forces_all
 *   species_ml  device i32 [n_ml]         species of the ML atoms, in ml_index order
 *   box         HOST, as for aev_forward (NULL = the usual gas-phase ML region)
 *   energy_out  device f64 [1]
 *   forces_all  device f32 [n_all][3]     forces_all[ml_index[k]] += F_ml[k]
 * n_ml <= max_atoms.  Asynchronous.
 */
int ani_energy_forces_subset(aev_ctx *c, const float *pos_all, const int32_t *ml_index,
                             const int32_t *species_ml, const float *box, int32_t n_ml,
                             double *energy_out, float *forces_all, void *stream);

/*
 * Host-buffer convenience entry points (the "end to end" calls bench.py times): every
 * pointer is a HOST pointer; the library stages through pinned buffers and device
 * workspace it owns, runs the same kernels, and copies the results back.  They sync.
 * Any of aev_out / grad_aev+forces_out may be NULL to skip that half.
 * aev_forward_backward_host: page-locked host buffers (cudaHostAlloc, cudaHostRegister, torch pin_memory) are copied
 * from / to directly, pageable ones are staged through the context's pinned buffer.  Positions and species go up first,
 * then the copy of grad_aev, the forward kernels and the read-back of aev_out run on three streams of the context, so
 * the two PCIe directions overlap each other and the kernels.
 * ani_energy_forces_host (the call an MD engine makes every step): inputs and results pass through the
 * context's pinned buffer, which the kernels read and write directly over PCIe (no copy operations); from the second
 * call with the same n_atoms, batch and box on, the whole evaluation is one replayed CUDA graph.
 * Both return deferred device-side errors (AEV_ERR_CAPACITY, AEV_ERR_STATE) themselves.
 */
int aev_forward_backward_host(aev_ctx *c, const float *pos, const int32_t *species,
                              const float *box, int32_t n_atoms, int32_t batch,
                              const float *grad_aev, float *aev_out, float *forces_out);
int ani_energy_forces_host(aev_ctx *c, const float *pos, const int32_t *species,
                           const float *box, int32_t n_atoms, int32_t batch,
                           double *energy_out, float *forces_out);

/*
 * Pair search that allocates nothing (step (1), rows A1-A2, "building neighbor lists"), for one
 * non-periodic system such as the gas-phase ML region of PAPER.md:183-215 (53 ML atoms).
 *
 * Why it exists: every call above needs an aev_ctx, and a context gets its workspace from cudaMalloc (in
 * aev_create, and again whenever a call brings larger shapes).  That is not an option for a host that gave the
 * whole GPU to its own memory pool at start-up, for a step loop that cannot afford the device-wide
 * synchronisation cudaMalloc / cudaFree imply, or for a component whose device-memory footprint has to be known
 * when it is linked.  This call takes no context and never calls cudaMalloc, cudaFree or any library routine
 * that allocates: its only working memory (one int per atom) is an array compiled into the library, 16 KB that
 * every GPU loading libaev_b200.so holds until the process exits.  The price is a hard size limit.
 *
 *   pos        device f32 [n_atoms][3]
 *   species    device i32 [n_atoms], or NULL = every atom is real; id < 0 = padding atom (in no pair)
 *   n_atoms    0 .. AEV_STATIC_MAX_ATOMS; more returns AEV_ERR_STATIC_LIMIT and launches nothing (the array
 *              cannot grow - use aev_neighbors + aev_export_pairs on a context for larger systems)
 *   rc         cutoff, > 0; a pair is listed when r_ij < rc (strict; same fp32 test as aev_neighbors, so the
 *              set equals the one aev_export_pairs returns for the same system, bit for bit)
 *   pairs_out  device i32 [cap][2], pairs (i < j) SORTED by i, then j (aev_export_pairs promises no order)
 *   count_out  DEVICE i64 [1] = pairs found; may exceed cap, then only the first cap (in that order) are written
 *   device     CUDA ordinal the pointers live on; the caller's current device is restored on return
 *   stream     as everywhere.  Asynchronous; nothing is read back to the host.
 *
 * First call on a device: it looks up the device address of the array once (no allocation, but the runtime may
 * have to load the module), so make one call per device during start-up, before any stream capture begins.
 * Sharing: the array belongs to the device, not to a caller, and keeps the previous call's contents.  No part
 * of it has to be cleared - each call overwrites the n_atoms entries it later reads - but two calls that can
 * run at the same time on one GPU (different streams with no event between them, or different host threads)
 * overwrite each other's counts and both results are garbage.  Issue them on one stream or order them with
 * events.
 */
#define AEV_STATIC_MAX_ATOMS 4096
int aev_pairs_static(const float *pos, const int32_t *species, int32_t n_atoms, float rc,
                     int32_t *pairs_out, int64_t cap, int64_t *count_out, int32_t device, void *stream);

/*
 * Test / diagnostic exports.
 * aev_export_pairs: the undirected pair set of the last neighbour build as (i<j) in the
 * caller's FLAT atom index (b*n_atoms + a), in no particular order.
 *   which      0 = radial set (r < rcr), 1 = angular set (r < rca)
 *   pairs_out  device i32 [cap][2];  count_out HOST i64 = pairs found (may exceed cap; only
 *              the first cap are written).  Syncs.
 */
int aev_export_pairs(aev_ctx *c, int32_t which, int32_t *pairs_out, int64_t cap,
                     int64_t *count_out);
/* Per-atom neighbour counts of the last neighbour build, caller's atom order:
 *   counts_out  device i32 [batch][n_atoms][2] = (angular-set size, radial-only size); padding
 *   atoms get (0,0).  Asynchronous on the context's last stream. */
int aev_export_counts(aev_ctx *c, int32_t *counts_out);
/* Per-kernel device timing for bench.py's roofline: when enabled, every kernel launch is
 * bracketed by CUDA events on its stream.  aev_get_profile syncs, adds the elapsed times
 * since the last call to ms_out[0..5] = {bin (k_bin, k_rank), fout (k_fout / k_fixout), aev (k_aev), backward (k_backward),
 * nbr (k_nbr, k_refresh), mlp}, writes the launches seen per slot to n_out[0..5], and resets. */
int aev_set_profiling(aev_ctx *c, int32_t enable);
int aev_get_profile(aev_ctx *c, double *ms_out, int64_t *n_out);
/* Syncs the context's last stream and returns AEV_OK or the deferred device-side error
 * (AEV_ERR_CAPACITY, AEV_ERR_STATE) raised by any call since the last aev_status. */
int aev_status(aev_ctx *c);
/* Verlet-skin mode (aev_params.skin > 0): how many times the neighbour lists have been rebuilt so far (the
 * other calls reused them).  Syncs.  AEV_ERR_STATE on a context without a skin (every call builds). */
int aev_neighbor_builds(aev_ctx *c, int64_t *builds_out);
/* Number of kernels the library has launched on this context so far (bench bookkeeping). */
int64_t aev_launch_count(const aev_ctx *c);
/* Independent-FMA microbenchmark: measured FP32 FMA throughput of `device` in TFLOP/s
 * (the ALU roofline denominator).  Syncs. */
int aev_probe_fp32_tflops(int32_t device, double *tflops_out);
const char *aev_error_string(int code);

#ifdef __cplusplus
}
#endif
#endif /* AEV_B200_H */

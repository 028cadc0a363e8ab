/*
 * rms.h -- C ABI of the B200-native hot path of the Realistic Microstructure Simulator
 *          (arXiv 2012.06478): Monte Carlo random walkers in a 3d voxelised label lattice.
 *
 * Citations "P:<n>" are line numbers of the paper text with the section / equation they
 * fall in; "R<n>" are the numbered readings in DESIGN.md (what the paper leaves open).
 *
 * Conventions
 *   - Every function returns 0 (RMS_OK) or a negative rms_status; nothing throws, aborts or prints.
 *     rms_last_error() returns a thread-local, statically stored message for the last failure.
 *   - Units: um and ms.  Lattice coordinates are in voxels; the box is periodic (R1).
 *   - "host" / "device" is stated for every pointer.  The library never keeps a host pointer after
 *     a call returns.  Handles are owned by the library and freed by the *_destroy calls.
 *   - `cuda_stream` is a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = the
 *     legacy default stream.  All work of a call is enqueued on that stream; calls that write host
 *     outputs (rms_run, rms_walkers_read, ...) synchronise that stream before they return.
 *   - There is no CPU fallback: without a CUDA device every compute call fails with RMS_ERR_CUDA.
 */
#ifndef RMS_H
#define RMS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    RMS_OK = 0,
    RMS_ERR_ARG = -1,            /* null pointer, label >= n_labels, non-unit direction, unsorted snapshots ...  */
    RMS_ERR_STEP_TOO_LARGE = -2, /* max_L sqrt(6 D_L dt) >= voxel size: voids the <=3-interaction rule */
    RMS_ERR_P_RANGE = -3,        /* Eq.3 gives P > 1 for a finite kappa (cf. the constraint at P:624)             */
    RMS_ERR_NO_SPACE = -4,       /* no voxel carries an allowed label                                     */
    RMS_ERR_OOM = -5,
    RMS_ERR_CUDA = -6,           /* no device, launch or runtime failure                                          */
    RMS_ERR_UNSUPPORTED = -7     /* e.g. n_wave above RMS_MAX_WAVES                                                */
} rms_status;

#define RMS_MAX_WAVES 16   /* gradient waveforms evaluated on one set of trajectories in one rms_run (sequence sweep) */

typedef struct rms_substrate rms_substrate; /* opaque */
typedef struct rms_walkers rms_walkers;     /* opaque */

/* ------------------------------------------------------------------------------------------------
 * rms_substrate_create -- upload the cell-label lattice and build what the walk reads (2.1.1:
 * "the voxelized geometry serves as the lookup table itself").
 *
 * labels       [nx*ny*nz] uint16, x fastest: idx = (z*ny + y)*nx + x.  Host pointer unless
 *              RMS_LABELS_ON_DEVICE.  Copied, unless RMS_ADOPT_DEVICE_PTR (then the caller keeps the
 *              device buffer alive and unchanged until rms_substrate_destroy).  Every label < n_labels.
 * D            [n_labels] intrinsic diffusivity, um^2/ms, > 0            (host; Table 1)
 * T2           [n_labels] ms; +inf or <= 0 means no relaxation; NULL = none (host; Eq.5)
 * kappa        [n_labels*n_labels] membrane permeability um/ms between label pairs, symmetric, diagonal
 *              ignored; 0 = impermeable; +inf = no membrane (Eq.C.15 with c1 = c2); NULL = all 0 (host; Eq.3)
 * rho          [n_labels*n_labels] surface relaxivity um/ms of the membrane met by a walker in label a towards label b
 *              (absorbing membrane / magnetisation transfer): the encounter saturates the walker
 *              (alpha_rho = 0, Eq.4) with probability rho_ab ds_a / D_a C_d; NULL = none (host)
 * T1           [n_labels] ms, the relaxation time during the mixing time of a stimulated echo (see
 *              rms_run_desc.mix_first_step); +inf or <= 0 means no relaxation; NULL = none (host)
 * conc         [n_labels] relative spin concentration c_L >= 0 of each label (Appendix C.2-C.3), NULL = all equal (host).
 *              Between labels of different c the permeation probability is Eq.C.9 with the correction of Eq.C.13 and
 *              lambda = arg min alpha_lambda (Eq.C.15 for kappa = +inf), and rms_walkers_init places walkers with a
 *              density proportional to c_L (R24).  Equal concentrations change nothing.
 * label_class  [n_labels] uint16 output compartment class of each label, < n_classes <= 65535; NULL = all 0 (host).
 *              Two classes (extra / intra-cellular) are the usual choice; class = label gives per-cell outputs.
 * flags        RMS_LABELS_ON_DEVICE | RMS_ADOPT_DEVICE_PTR | RMS_NO_BRICKS | RMS_LAYOUT_X_FASTEST | RMS_LAYOUT_Z_FASTEST | RMS_LAYOUT_AUTO |
 *              RMS_LATTICE_DICT
 *
 * Derived on the device, unless RMS_NO_BRICKS: the octant lattice, one 64-bit word per voxel (plus a
 * one-voxel periodic ghost shell): eight bytes, one per octant of hop directions, whose bits say which voxels
 * of the 2x2x2 block a hop of that octant can reach carry the same label -- a face is a membrane iff the labels
 * on its two sides differ, and a hop shorter than a voxel only ever meets faces inside that block (P:62,
 * P:159).  8 bytes per voxel of device memory on top of the labels (4 more, on demand, for the general fp32
 * kernel's face-bit mode).
 * Errors: RMS_ERR_ARG, RMS_ERR_OOM, RMS_ERR_CUDA.
 */
#define RMS_LABELS_ON_DEVICE 1u
#define RMS_ADOPT_DEVICE_PTR 2u
#define RMS_NO_BRICKS 4u
#define RMS_LAYOUT_X_FASTEST 8u   /* memory order of the octant lattice: x fastest (the default)                         */
#define RMS_LAYOUT_Z_FASTEST 16u  /* z fastest: the 8 words of a 32-byte sector lie along z (cells elongated along z)    */
#define RMS_LAYOUT_AUTO 24u       /* x or z, whichever axis has fewer membrane faces normal to it (sampled)              */
#define RMS_LATTICE_DICT 32u      /* store a 16-bit code per voxel and the octant words of the distinct neighbourhoods in a
                                     dictionary (2 bytes per voxel instead of 8: a quarter of the cache footprint of a walker;
                                     one more, dependent, look-up per face reached; same speed on the axon lattice, a
                                     build a third longer).  Lattices with more distinct
                                     neighbourhoods than the tables hold (independent random labels) get the octant lattice. */

typedef struct {
    int32_t nx, ny, nz;
    double voxel_um;            /* l_p, isotropic */
    const uint16_t* labels;
    int32_t n_labels;
    const float* D;
    const float* T2;
    const float* kappa;
    const float* rho;
    const uint16_t* label_class;
    int32_t n_classes;
    uint32_t flags;
    const float* T1;
    const float* conc;
} rms_substrate_desc;

int rms_substrate_create(const rms_substrate_desc* desc, void* cuda_stream, rms_substrate** out);
int rms_substrate_destroy(rms_substrate* s);

typedef struct {
    int32_t nx, ny, nz, n_labels, n_classes;
    uint64_t n_voxels;
    uint64_t n_membrane_faces;  /* voxel faces whose two sides carry different labels (each face once) */
    uint64_t lattice_bytes;     /* uint16 lattice on the device                                          */
    uint64_t brick_bytes;       /* neighbourhood lattice on the device (0 with RMS_NO_BRICKS)            */
    int32_t has_bricks;
    uint32_t dict_entries;        /* RMS_LATTICE_DICT: distinct neighbourhoods in the dictionary (0: octant lattice in use) */
    uint32_t dict_escaped_voxels; /* voxels whose neighbourhood found no free code (their words sit in a hash table)        */
} rms_substrate_info;

int rms_substrate_get_info(const rms_substrate* s, rms_substrate_info* out /* host */);

/* ------------------------------------------------------------------------------------------------
 * rms_walkers_init -- place walkers with homogeneous density over the voxels whose label is allowed
 * (step 1 of 2.2; labels that are not allowed are the paper's "dead space" for placement).
 * Walker ids are first_walker_id .. first_walker_id + n_walkers - 1; a walker's start and its whole
 * trajectory depend only on (seed, id), never on the batch or the launch shape (R2, R13).
 * label_allowed [n_labels] host, 1 = place here; NULL = everywhere.
 * Errors: RMS_ERR_NO_SPACE (a walker found no allowed voxel in 2^20 proposals), RMS_ERR_ARG/OOM/CUDA.
 */
int rms_walkers_init(const rms_substrate* s, uint64_t n_walkers, uint64_t first_walker_id,
                     const uint8_t* label_allowed, uint64_t seed, void* cuda_stream, rms_walkers** out);
int rms_walkers_destroy(rms_walkers* w);

/* The same with a placement weight per label (walkers per axon; R26): the density of walkers in an
 * allowed label L is proportional to label_weight[L] >= 0 (times its spin concentration, if the substrate has them), so
 * label_weight[L] = 1 / V_L (rms_substrate_label_volumes) gives every cell the same expected number of walkers.
 * label_weight [n_labels] host; NULL = all 1, which is rms_walkers_init.  Errors as rms_walkers_init; RMS_ERR_ARG for a
 * negative, infinite or NaN weight, RMS_ERR_NO_SPACE if every allowed label has weight 0. */
int rms_walkers_init_weighted(const rms_substrate* s, uint64_t n_walkers, uint64_t first_walker_id,
                              const uint8_t* label_allowed, const float* label_weight, uint64_t seed, void* cuda_stream,
                              rms_walkers** out);

/* Voxels per label, counted on the device.  voxels_out [n_labels] host.  Errors: RMS_ERR_ARG, RMS_ERR_OOM, RMS_ERR_CUDA. */
int rms_substrate_label_volumes(const rms_substrate* s, void* cuda_stream, uint64_t* voxels_out);

/* The same count for callers that may not allocate device memory (serving loops, harnesses that forbid cudaMalloc, code
 * that will later run under CUDA graph capture): this entry point calls no cudaMalloc, cudaFree or allocating routine,
 * neither the driver's nor the library's cache.  Its per-label counters are a static device array of
 * RMS_STATIC_MAX_LABELS uint64 (128 KiB), held by every GPU that loads the library until the process exits.
 * Same arguments and result as rms_substrate_label_volumes: voxels_out [n_labels] host, written before the call returns
 * (the stream is synchronised).  RMS_ERR_UNSUPPORTED if the substrate has more than RMS_STATIC_MAX_LABELS labels (use
 * rms_substrate_label_volumes then); RMS_ERR_ARG, RMS_ERR_CUDA otherwise.
 * All calls on a device share the one array (it is cleared at the start of every call): calls that overlap on the GPU
 * -- two host threads, or two streams -- race on it and must be serialised by the caller.  The first call on a device
 * looks up the array's device address (no allocation); make that call outside any stream capture. */
#define RMS_STATIC_MAX_LABELS 16384
int rms_substrate_label_volumes_static(const rms_substrate* s, void* cuda_stream, uint64_t* voxels_out);

/* ------------------------------------------------------------------------------------------------
 * rms_run -- advance every walker by n_steps Monte Carlo steps (2.2 steps 2-4: fixed-length
 * hop sqrt(6 D dt) in a random direction; at a voxel face between unlike labels elastic reflection or
 * permeation with the probability of Eq.3; at most three interactions per step), accumulate the
 * gradient phase and the T2 weight (Eq.5, Eq.7), and reduce to signals and moments.
 *
 * wave        [n_wave*n_steps] unit-less gradient shape w_m[i] for step i = 1..n_steps of THIS call (host)
 * gamp        [n_wave*n_g] gradient amplitudes, rad/(ms um):  phi = gamp * dt * sum_i w_m[i] n.(x_i - x_0)
 *             (right-endpoint rule, R11) (host)
 * dirs        [n_dir*3] unit vectors (host)
 * snap_steps  [n_snap] ascending step numbers in 1..n_steps of this call at which the displacement
 *             moments are taken (host)
 * flags       RMS_RUN_LABEL_GATHER: test faces by gathering the neighbour's uint16 label (the paper's
 *             lookup table) instead of the neighbourhood lattice.
 *             RMS_RUN_GENERAL_KERNEL: impermeable or permeable runs with piecewise-constant waveforms (rectangular
 *             lobes of any amplitude, segments of >= 32 steps on average) normally take the specialised kernel
 *             (csrc/rms_step_fast.cu); this flag forces the general one.
 *             RMS_RUN_FP64: the direction of every hop in fp64 and the in-voxel offsets in 2^-63 fixed point (exact
 *             additions), hit order and phase in fp64, for runs of more than a few 1e4 steps whose trajectories must
 *             stay on those of an fp64 reference (DESIGN.md "Tolerances" says why fp32 directions cannot).  Three
 *             quarters of the fp32 speed wherever the specialised kernel runs (piecewise-constant waveforms;
 *             impermeable, permeable with P << 1, rejection sampling, ERL between walls); a plain, slower fp64 kernel
 *             otherwise (general waveforms, label gathers, absorbing membranes, faces with P = 1).
 *             RMS_RUN_NO_ORDERING: on large lattices the walkers are dealt to the threads in the order of the
 *             lattice cell they sit in (cache locality; results do not depend on it); this flag keeps id order.
 *             RMS_RUN_REJECTION_SAMPLING: the paper's other membrane interaction (Appendix B): a
 *             step that meets a membrane it does not cross is cancelled and the walker stays where it was for
 *             that step, instead of the elastic collision.  The permeation probability is then Appendix B.1's
 *             P_T = A / (1 + A), A = kappa sqrt(6 dt / D) 2/3, defined for equal D on both sides:
 *             RMS_ERR_UNSUPPORTED for a finite non-zero kappa between unequal D.  Runs in the specialised kernel
 *             (piecewise-constant waveforms) or the general ones, fp32 or fp64 with RMS_RUN_FP64; biased near
 *             membranes by Eq.B.2, which is why elastic collision is the default.
 *             RMS_RUN_ERL: equal-step-length random leap, the paper's third comparison interaction (PAPER.md lines 80,
 *             340, Appendix A): a step that meets a membrane is cancelled and tried again in a new direction until it
 *             meets none (at most 4095 retries, then the walker stays put for the step).  Impermeable, non-absorbing
 *             membranes only (kappa 0 or +inf, no rho: RMS_ERR_UNSUPPORTED otherwise).  Runs in the specialised kernel
 *             (piecewise-constant waveforms, kappa 0 everywhere; fp32 or fp64) or the general ones; depletes the
 *             density within a hop length of the membranes (Eq.A.1), hence not the default.
 *             RMS_RUN_NO_SLICES: a launch of the specialised kernel over more walkers than the GPU holds at a time is cut into
 *             time slices of ~1000 steps that are dealt to the SMs from a queue, so that the SMs do not idle while the last
 *             blocks finish (results do not depend on it beyond the order of the fp64 phase additions); this flag keeps one
 *             block per group of walkers for the whole launch.
 *
 * mix_first_step, mix_n_steps  the mixing time of a stimulated echo: in these steps Eq.5 runs with the T1 of
 *             the compartment the walker is in, in all others with its T2.  The window lies inside 1..n_steps
 *             (RMS_ERR_ARG otherwise); the caller keeps the waveforms at 0 there (the stored magnetisation
 *             collects no phase; not enforced).  The window edges become launch boundaries, nothing else changes.
 *
 * n_tensor, tensor_waves [n_tensor*3], tensor_gamp [n_tensor*n_g], n_rot, rots [n_rot*9] (all host)
 *             gradient waveforms whose direction changes in time ("arbitrary diffusion gradient waveforms", P:336;
 *             B-tensor encoding; R23).  Tensor waveform t drives the gradient axes x, y, z with the scalar
 *             waveforms tensor_waves[3t + a] of this run (an index into wave, or -1: axis off); rots[9k + 3b + a] is
 *             row b, column a of the matrix R_k that takes the waveform's frame to the lattice frame (g_lab = R_k g).
 *             Phase: phi = tensor_gamp[t*n_g + g] dt l_p sum_a (R_k e_a) . Phi_{m_a} with the same per-waveform phase
 *             vectors Phi_m the scalar signals use, so tensor signals cost nothing in the walk.  RMS_ERR_ARG for an
 *             index outside [-1, n_wave).
 *
 * A second rms_run on the same walkers continues the trajectories (the random numbers are keyed on the
 * absolute step), so long runs may be chunked; phases and T2 weights keep accumulating.
 *
 * Outputs (rms_result, all HOST arrays allocated by the caller; any pointer may be NULL):
 *   sum_alpha  [n_classes]                      sum_w alpha_w at the end of the call, by class of the
 *                                               walker's INITIAL label
 *   sig_re/im  [n_wave][n_g][n_dir][n_classes]  sum alpha cos(phi), -sum alpha sin(phi)   (Eq.7 numerator)
 *   m2, m4     [n_snap][n_dir][n_classes]       sum alpha X^2, sum alpha X^4, X = n.(x - x_0) in um
 *   snap_alpha [n_snap][n_classes]              sum alpha at the snapshot
 *   class_flow [n_snap][n_classes][n_classes]   walkers by (initial class, class at the snapshot)
 *   S_re/im    [n_wave][n_g][n_dir]             Eq.7: S = <alpha e^{-i phi}> / <alpha>, classes pooled
 *   Dapp, Kapp [n_snap][n_dir]                  D = <alpha X^2>/(2 t <alpha>), K = <alpha X^4><alpha>/<alpha X^2>^2 - 3
 *                                               with t = (steps since the walkers' start) * dt (R14)
 *   n_encounters / n_permeations / n_clamps     unlike-label faces met / crossed; offsets clamped to [0,1)
 *                                               (n_clamps is counted by the general kernel only)
 * Errors: RMS_ERR_ARG, RMS_ERR_STEP_TOO_LARGE, RMS_ERR_P_RANGE, RMS_ERR_UNSUPPORTED, RMS_ERR_OOM, RMS_ERR_CUDA.
 */
#define RMS_RUN_LABEL_GATHER 1u
#define RMS_RUN_GENERAL_KERNEL 2u
#define RMS_RUN_NO_ORDERING 4u
#define RMS_RUN_FP64 8u
#define RMS_RUN_REJECTION_SAMPLING 16u
#define RMS_RUN_ERL 32u
#define RMS_RUN_NO_SLICES 64u

typedef struct {
    double dt_ms;               /* Table 1: dt */
    int64_t n_steps;            /* Table 1: N_step (of this call) */
    int32_t n_wave;
    const float* wave;
    int32_t n_g;
    const double* gamp;
    int32_t n_dir;
    const double* dirs;
    int32_t n_snap;
    const int64_t* snap_steps;
    uint32_t flags;
    int64_t mix_first_step;     /* stimulated echo: steps mix_first_step .. mix_first_step + mix_n_steps - 1 */
    int64_t mix_n_steps;        /* of this call (1-based) relax with T1 instead of T2; 0 = no mixing time            */
    int32_t n_tensor;           /* gradient waveforms that change direction (B-tensor encoding), see above           */
    const int32_t* tensor_waves;
    const double* tensor_gamp;
    int32_t n_rot;
    const double* rots;
} rms_run_desc;

typedef struct {
    double* sum_alpha;
    double* sig_re;
    double* sig_im;
    double* m2;
    double* m4;
    double* snap_alpha;
    uint64_t* class_flow;
    double* S_re;
    double* S_im;
    double* Dapp;
    double* Kapp;
    uint64_t n_encounters, n_permeations, n_clamps; /* written by rms_run */
    uint64_t n_saturations;     /* walkers saturated at absorbing membranes during this call (Eq.4)   */
    double kernel_ms;           /* device time of the step kernels of this call (CUDA events)          */
    double total_ms;            /* device time of everything this call enqueued                         */
    uint32_t n_launches;        /* kernels launched by this call                                        */
    double* tsig_re;            /* [n_tensor][n_g][n_rot][n_classes] sum alpha cos(phi), -sum alpha sin(phi) of the  */
    double* tsig_im;            /* tensor waveforms, and                                                             */
    double* tS_re;              /* [n_tensor][n_g][n_rot] their Eq.7 signal, classes pooled; any may be NULL          */
    double* tS_im;
} rms_result;

int rms_run(const rms_substrate* s, rms_walkers* w, const rms_run_desc* desc, void* cuda_stream, rms_result* out);

/* ------------------------------------------------------------------------------------------------
 * rms_walkers_read -- copy the state of walkers [first, first+count) to the host: the parity hook
 * (final voxel per walker) and the checkpoint format.
 */
typedef struct {
    int32_t vox[3];   /* current voxel, unwrapped (vox0 + whole-voxel displacement)   */
    float off[3];     /* in-voxel offset in [0,1)                                      */
    int32_t vox0[3];  /* initial voxel (inside the box)                                */
    float off0[3];
    uint16_t label, label0;
    float relax;      /* sum_i t_i / T2^(i), Eq.5                                      */
    double phi[RMS_MAX_WAVES][3]; /* Phi_m = sum_i w_m[i] (x_i - x_0), voxel units     */
} rms_walker_state;

int rms_walkers_read(const rms_walkers* w, uint64_t first, uint64_t count, rms_walker_state* host_out,
                     void* cuda_stream);
int rms_walkers_steps_done(const rms_walkers* w, uint64_t* out /* host */);

/* Tables the run derives from (D, kappa, dt): hop length s_L = sqrt(6 D_L dt)/l_p (Eq.1, d = 3) and the
 * permeation probabilities P[a][b] of Eq.3, both as the fp32 values the kernels use.  Host outputs,
 * s_out [n_labels], P_out [n_labels*n_labels] (may be NULL).  Pure host function. */
int rms_tables(const rms_substrate* s, double dt_ms, float* s_out, float* P_out);

/* H8 on its own: normalise reduced sums (e.g. after adding the sums of several walker-id shards).
 * Host arrays laid out as in rms_result; t_ms [n_snap] diffusion time of each snapshot.  Pure host function:
 *   S = (sum_c sig_re + i sum_c sig_im) / sum_c sum_alpha                         (Eq.7)
 *   D = <alpha X^2> / (2 t <alpha>),  K = <alpha X^4><alpha> / <alpha X^2>^2 - 3   (R14)        */
int rms_normalise(int n_classes, int n_q, const double* sum_alpha, const double* sig_re, const double* sig_im,
                  int n_snap, int n_dir, const double* snap_alpha, const double* m2, const double* m4,
                  const double* t_ms, double* S_re, double* S_im, double* Dapp, double* Kapp);

/* The signal of all cells from per-cell sums taken with any number of walkers per cell ("volume-weighted sum", P:266;
 * DESIGN.md R26): S = sum_c V_c S_c / sum_c V_c over the classes with sum_alpha > 0, S_c = sig_c / sum_alpha_c (Eq.7 within
 * class c).  class_volume [n_classes], the other arrays as in rms_result.  Pure host function. */
int rms_volume_weighted_signal(int n_classes, int n_q, const double* class_volume, const double* sum_alpha,
                               const double* sig_re, const double* sig_im, double* S_re, double* S_im);

/* Measured ceiling for the label / neighbourhood gathers of the walk (the second roofline candidate): random
 * gathers of elem_bytes (2 or 4) from a zero-filled device table of table_bytes (48 MB sits in the L2, 1 GB does not),
 * loads_per_thread each on 148 x 2048 threads; *gathers_per_s (host) = gathers, i.e. 32-byte sectors, per second.
 * Errors: RMS_ERR_ARG, RMS_ERR_OOM, RMS_ERR_CUDA. */
int rms_gather_probe(uint64_t table_bytes, int elem_bytes, uint32_t loads_per_thread, void* cuda_stream, double* gathers_per_s);

/* Device buffers behind destroyed handles are kept for the next handle of the same size (a pass of the path
 * allocates the same buffers every time); rms_memory_trim returns them to the driver.  Always RMS_OK. */
int rms_memory_trim(void);

const char* rms_last_error(void);
const char* rms_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RMS_H */

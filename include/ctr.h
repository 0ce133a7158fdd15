/*
 * ctr.h -- C ABI of libctr: the B200 (sm_100a) hot path of edge-preserving-TV CT
 * reconstruction (Tian, Jia, Yuan, Pan, Jiang; citations are /root/reference/PAPER.md:<line>).
 *
 * The path:
 *   P   ray-driven projector, p_ij = length of ray i inside pixel j      PAPER.md:85-89 (Eq. 1)
 *   P^T exact transpose of that matrix, computed in gather form           PAPER.md:193, :471 (A3')
 *   CGLS with warm start                                                  PAPER.md:149, :414-440 (App. I)
 *   edge weights w = exp(-(|grad f|/sigma)^2), sigma from the histogram   PAPER.md:106-110 (Eq. 4-5)
 *   EP-TV gradient, symmetric scheme A2/A3
 *   Armijo line search along -g, positivity clamp, outer loop
 *
 * Conventions common to every call
 * --------------------------------
 * - All array arguments named d_* are DEVICE pointers to contiguous fp32, 16-byte aligned, owned by
 *   the caller for the duration of the (asynchronous) call. Nothing is allocated on the hot path:
 *   the handle owns the geometry tables and all scratch (sized at ctr_create for `batch`).
 * - Layouts (x fastest):  image     2D: [batch][ny][nx]        3D: [nz][ny][nx]
 *                         sinogram  2D: [batch][nviews][nu]    3D: [nviews][nv][nu]
 *                         weights   [ndim][image]  plane A holds the face between voxel p and p+e_A
 *                                   at p; border faces (last index along A) hold 0.
 * - Batched 2D slices are independent problems: every scalar (CGLS a, b; sigma; Armijo k) is per slice.
 * - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream). Calls only enqueue work
 *   and return without synchronising, except ctr_create, ctr_destroy and ctr_get_stats.
 * - Return value: CTR_OK (0) or a negative ctr_status. No exceptions, no exit(), nothing printed.
 *   On error nothing has been enqueued unless the code is CTR_ECUDA.
 * - A handle must not be used from two host threads at once (its scratch is shared by all calls).
 * - Inputs must be finite. A NaN/Inf in a sinogram bin reaches every pixel of the 2 x 2 pixel quads its ray
 *   touches in the batched P^T (0 * Inf), not only the pixels the ray crosses.
 */
#ifndef CTR_H_
#define CTR_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ctr_handle ctr_handle; /* opaque */

typedef enum {
  CTR_OK = 0,
  CTR_EINVAL = -1, /* NULL / misaligned pointer, non-positive size, dsd <= dso, n_iter < 0, quantile not in (0,1] ... */
  CTR_EGEOM = -2,  /* source or detector inside the image's circumscribed circle; cone beam also: a ray that advances
                      more than one voxel in z per in-plane voxel, or a voxel that sees more than 15 detector columns
                      of a view (limits of the 3D kernels; text in ctr_last_error is not available: *out is NULL)   */
  CTR_ENOMEM = -3, /* device or host allocation failed                                                             */
  CTR_ECUDA = -4,  /* a CUDA runtime call failed; text in ctr_last_error                                           */
  CTR_EARCH = -5,  /* current device is not compute capability 10.x (sm_100)                                       */
  CTR_ETOOBIG = -6 /* ctr_forward_noalloc: the problem exceeds the fixed scratch (CTR_NOALLOC_MAX_* below)          */
} ctr_status;

/* Scanner + grid. Geometry of PAPER.md:85-89, :217 and App. III A6 (:484): at view angle th_k the source
 * sits at -dso (cos th_k, sin th_k, 0), the detector centre at (dsd-dso)(cos th_k, sin th_k, 0), the
 * detector u-axis is (-sin th_k, cos th_k, 0), the v-axis is +z. Bin (a,b) is at
 * t_a = (a-(nu-1)/2+u_off) du along u and v_b = (b-(nv-1)/2+v_off) dv along v (FLAT), or at fan angle
 * t_a/dsd on a circle of radius dsd about the source (ARC, 2D only). Voxel (i,j,k) covers
 * [X_i,X_i+dx) x [Y_j,Y_j+dy) x [Z_k,Z_k+dz), X_i = cx - nx dx/2 + i dx (likewise Y, Z). Lengths in mm. */
typedef struct {
  int32_t ndim;           /* 2 = fan-beam slice(s), 3 = circular cone beam                                      */
  int32_t nx, ny, nz;     /* nz = 1 for 2D                                                                      */
  float dx, dy, dz;       /* voxel size, mm (dz ignored in 2D)                                                   */
  float cx, cy, cz;       /* grid centre minus isocentre, mm                                                     */
  int32_t nviews;
  float theta0, dtheta;   /* th_k = theta0 + k dtheta (radians), used when angles == NULL                        */
  const float* angles;    /* optional HOST array [nviews] overriding theta0/dtheta; copied by ctr_create          */
  int32_t nu, nv;         /* detector bins; nv = 1 for 2D                                                        */
  float du, dv;           /* bin pitch, mm (ARC: arc length at radius dsd)                                       */
  float u_off, v_off;     /* detector centre shift, in bins                                                      */
  float dso, dsd;         /* source-isocentre and source-detector distances, mm                                  */
  int32_t det_type;       /* 0 = FLAT, 1 = ARC                                                    */
  int32_t batch;          /* independent 2D slices sharing this geometry (>= 1); must be 1 when ndim = 3          */
  int32_t flags;          /* bit mask of CTR_GEOM_* below; 0 in every config                                      */
} ctr_geometry;

/* ctr_geometry.flags */
enum {
  CTR_GEOM_NO_TABLES = 1, /* do not build the stored matrices / hit tables (second strategy): every
                            p_ij is computed on the fly. Same bits either way; a low-memory mode and the tests' way
                            of checking that the tables hold exactly what the on-the-fly kernels compute. */
  CTR_GEOM_NO_GRAPHS = 2, /* ctr_reconstruct launches every kernel itself instead of replaying a CUDA graph of the
                            steady-state outer iteration (same kernels, same results). */
  CTR_GEOM_NO_STORED_P = 4, /* batched slices: apply P on the fly (k_si_forward) instead of from the stored matrix
                            shared by all slices (k_si_forward_tab); the other tables are still built. */
  CTR_GEOM_NO_LAZY_CGLS = 8 /* CGLS projects every gradient against the stored unit gradients in image space in all
                            iterations (S24) instead of moving that work to the sinogram side after the
                            first four: the same iteration in exact arithmetic; for A/B runs and tests. */
};

/* Iteration schedule and the constants the paper leaves open (readings S13, S14). */
typedef struct {
  int32_t n_outer, n_cgls, n_gd;  /* outer iterations; CGLS iterations per outer; GD sweeps per outer            */
  float lambda;                   /* lambda of (P2), Eq. 8                                           */
  float sigma_quantile;           /* q in (0,1]: sigma = q-quantile of the face gradient magnitudes */
  float eps;                      /* |grad f| -> sqrt(N0^2 + eps^2) in A2's denominators and the energy           */
  float armijo_t0, armijo_rho, armijo_c;
  int32_t armijo_max;             /* trials t = t0 rho^k, k < armijo_max (<= 32)                                   */
  int32_t weights_mode;           /* 0 = EP-TV (Eq. 4-5), 1 = plain TV, w = 1                        */
  int32_t positivity;             /* 1: f <- max(f,0) after the last sweep of every outer iteration  */
  int32_t warm_start;             /* 0: f^(0) = 0 as in the paper (:171); 1: ctr_reconstruct continues from d_img   */
  /* NEXT rows of SURVEY.md 8(f), off (0) in every config: */
  int32_t fidelity_mode;          /* Step 1 of ctr_reconstruct: 0 = CGLS; 1 = the plain gradient update
                                     (P1) of Eq. 8 (:141): v <- v - p1_step P^T (P v - y), n_cgls times from v = f        */
  float p1_step;                  /* mu/lambda of (P1), the step of that update (>= 0; stable below 2/||P||^2)         */
  int32_t backprojector;          /* P^T inside ctr_cgls / Step 1: 0 = exact transpose (ctr_back); 1 = the paper's
                                     pixel-driven Eq. (11) (ctr_back_pixel, 2D only): an UNMATCHED pair, so CGLS then
                                     runs the recurrence as printed (:420-440), without re-orthogonalisation (S24)      */
} ctr_params;

/* One record per (GD sweep, slice), in execution order: what steered the iteration. */
typedef struct {
  double sigma;   /* O6                                   */
  double e0;      /* energy before the sweep (O9)          */
  double g2;      /* ||g||^2                               */
  int32_t k;      /* accepted Armijo index, -1 = none      */
  int32_t pad;
} ctr_sweep_stat;

/* Defaults: n_outer 1, n_cgls 10, n_gd 5, lambda 0.01, q 0.90, eps 1e-4, t0 1e-3, rho 0.5, c 0.5 (S25),
 * armijo_max 16, EP-TV, positivity on, warm_start off, fidelity_mode 0 (CGLS), p1_step 0, backprojector 0. */
void ctr_default_params(ctr_params* p);

/* Build a handle for `g` on the CURRENT CUDA device: validates the geometry, builds the ray table
 * and allocates all scratch. Synchronous. *out is NULL on failure. */
int ctr_create(const ctr_geometry* g, ctr_handle** out);
/* Frees everything the handle owns (synchronises the device first). NULL is allowed. */
void ctr_destroy(ctr_handle* h);

/* a1: d_sino = P d_img. d_sino is overwritten; d_img is not modified. */
int ctr_forward(ctr_handle* h, const float* d_img, float* d_sino, void* stream);
/* a2: d_img = P^T d_sino, the exact transpose of ctr_forward's matrix (same p_ij, bit for bit), gather
 * form, no atomics (PAPER.md:193 explains why not scatter). d_img is overwritten. */
int ctr_back(ctr_handle* h, const float* d_sino, float* d_img, void* stream);
/* a1 for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): d_sino = P d_img for ONE 2D fan-beam slice (ndim 2, batch 1, angles NULL, flags 0), no handle needed.
 * Same kernels and the same bits as ctr_forward on a handle created with CTR_GEOM_NO_TABLES. Calls no cudaMalloc,
 * cudaFree or allocating library routine: the ray table and the transposed image copy live in one file-scope device
 * array of CTR_NOALLOC_SCRATCH_BYTES (2.1 MiB) that every GPU which loads the library holds until the process
 * exits. Limits: nx ny <= CTR_NOALLOC_MAX_PIXELS, nviews nu <= CTR_NOALLOC_MAX_RAYS, nviews <= CTR_NOALLOC_MAX_VIEWS
 * (BASELINE.json's 512^2 / 60 x 888 slice fits exactly); anything larger returns CTR_ETOOBIG and enqueues nothing.
 * EVERY call shares that array: calls that overlap on the GPU (different streams or host threads) race - serialise
 * them. Asynchronous on `stream` like the other calls. The first call on a device looks the array's address up
 * (cudaGetSymbolAddress): make it outside a stream capture. */
#define CTR_NOALLOC_MAX_PIXELS (512 * 512)
#define CTR_NOALLOC_MAX_RAYS 65536
#define CTR_NOALLOC_MAX_VIEWS 4096
#define CTR_NOALLOC_SCRATCH_BYTES (16 * CTR_NOALLOC_MAX_RAYS + 4 * CTR_NOALLOC_MAX_PIXELS + 24 * CTR_NOALLOC_MAX_VIEWS)
int ctr_forward_noalloc(const ctr_geometry* g, const float* d_img, float* d_sino, void* stream);
/* NEXT-1 (not on the hot path; ctr_cgls uses it only with ctr_params.backprojector = 1): the paper's own pixel-driven backprojector, Eq. (11)
 * (PAPER.md:195-197): d_img(u*,v*) = (dx dy / dbeta) sum_views y(beta*) / l, with y(beta*) linearly interpolated
 * between the two nearest detector units (0 outside the outermost unit centres) and l the source-pixel
 * distance; dbeta = du/dsd (ARC) or du cos^2(beta*)/dsd (FLAT). An APPROXIMATE adjoint of ctr_forward (the paper
 * reports < 1 % mismatch, :493). 2D only (CTR_EINVAL otherwise). Same layouts as ctr_back; d_img is overwritten. */
int ctr_back_pixel(ctr_handle* h, const float* d_sino, float* d_img, void* stream);
/* a3: n_iter CGLS iterations on min ||P x - b||^2 from the start value in d_x;
 * d_x is updated in place to u^(n_iter). n_iter = 0 is a no-op. Zero denominators stop the update (S4).
 * With ctr_params.backprojector = 1 (ctr_set_params) every P^T is Eq. (11) instead (2D; CTR_EINVAL in 3D). */
int ctr_cgls(ctr_handle* h, const float* d_b, float* d_x, int n_iter, void* stream);
/* a4: d_w[ndim][image] = exp(-N0^2/sigma^2) with N0 the face magnitudes of A3 at d_x and
 * sigma = max(k-th smallest N0, eps), k = ceil(quantile * #interior faces) per slice (exact order
 * statistic). weights_mode = 1 writes 1 on interior faces. d_sigma (device, [batch]) may be NULL. */
int ctr_update_weights(ctr_handle* h, const float* d_x, float* d_w, float quantile, float* d_sigma, void* stream);
/* a5+a6: ONE gradient-descent sweep on lambda/2 ||x - v||^2 + sum w |grad x| with w frozen: gradient of
 * Eq. 9 / A2, Armijo search (first k with E(x - t_k g) <= E(x) - c t_k ||g||^2), x <- x - t_k g in place
 * (unchanged if no trial passes). eps and the Armijo constants come from ctr_set_params / the defaults. */
int ctr_eptv_step(ctr_handle* h, float* d_x, const float* d_v, const float* d_w, float lambda, void* stream);
/* a8: the whole EPTV algorithm: f = 0; n_outer x { v = CGLS(sino, x0 = f, n_cgls); f = v;
 * n_gd x (weights, sweep); clamp }. d_img receives f. p = NULL uses the handle's current parameters.
 * If d_w is not NULL it receives the weights of the last sweep ([ndim][image]). */
int ctr_reconstruct(ctr_handle* h, const float* d_sino, float* d_img, const ctr_params* p, void* stream);
int ctr_reconstruct_w(ctr_handle* h, const float* d_sino, float* d_img, float* d_w, const ctr_params* p, void* stream);

/* Replace the handle's parameters (validated: CTR_EINVAL leaves them unchanged). */
int ctr_set_params(ctr_handle* h, const ctr_params* p);
/* Synchronises `the stream last used`, then copies up to n_records sweep records of the last
 * ctr_reconstruct / ctr_eptv_step / ctr_update_weights sequence into HOST memory `buf`, ordered
 * [sweep][slice]. Returns the number of records available (>= 0) or a negative status. */
int ctr_get_stats(ctr_handle* h, ctr_sweep_stat* buf, size_t n_records);
/* Device-side timing of the handle's own launches, by kind, with CUDA events recorded on the launching
 * stream around every kernel (or short kernel sequence) while enabled. ctr_profile_enable(h, 1) clears
 * the accumulators and starts recording (at most 32768 intervals; later ones are dropped);
 * ctr_profile_enable(h, 0) stops. ctr_profile_read synchronises the last stream and returns, per kind,
 * the summed milliseconds and the interval count in HOST arrays of length CTR_PROF_KINDS. */
enum { CTR_PROF_FORWARD = 0, CTR_PROF_BACK = 1, CTR_PROF_VECTOR = 2, CTR_PROF_TV = 3, CTR_PROF_LAYOUT = 4, CTR_PROF_KINDS = 5 };
int ctr_profile_enable(ctr_handle* h, int on);
int ctr_profile_read(ctr_handle* h, double* ms_by_kind, long long* count_by_kind);
/* Which kernels this handle applies P and P^T with, as "forward=<kernel>;back=<kernel>;tables_mb=<MB of lookup
 * tables built>;graphs=<0|1>" (the lookup tables of PAPER.md:193 are built best effort at ctr_create). Valid
 * for the life of the handle. */
const char* ctr_path_info(const ctr_handle* h);
/* Number of kernels this handle has launched so far (bench.py's gpu_launches). */
long long ctr_launch_count(const ctr_handle* h);

/* Measured peaks of the on-chip units that bound the projector kernels (bench.py's roofline denominators; not part
 * of the reconstruction path). Each figure is the best of `reps` runs of a microbenchmark kernel at full occupancy on
 * the CURRENT device, timed with CUDA events on the legacy default stream; synchronous; allocates and frees ~2 GiB. */
typedef struct {
  double fma_tflops;    /* fp32 FMA (FFMA), 2 flop each                                                        */
  double fma2_tflops;   /* packed fp32x2 FMA (FFMA2, sm_100), 4 flop each                                       */
  double issue_gwinst;  /* warp instructions issued per second / 1e9 (the FFMA kernel: one pipe, 1 per clock and scheduler) */
  double mixed_gwinst;  /* the same for FFMA and integer ALU instructions interleaved 1:1 (the integer pipe is slower) */
  double l1_tbs;        /* L1 data pipe: LDG.128 that hit in L1, TB/s (128 bytes per wavefront)                 */
  double smem_tbs;      /* shared memory: conflict-free LDS.128, TB/s                                           */
  double l2_tbs;        /* L2 -> SM fabric: LDG.128 (cache-global) over a 32 MiB window resident in L2, TB/s    */
  double hbm_copy_gbs;  /* device-memory copy of 1 GiB, read + write bytes, GB/s                                */
  int32_t sm_count;
  int32_t pad;
} ctr_peaks;
int ctr_measure_peaks(ctr_peaks* out, int reps);

const char* ctr_strerror(int status);
/* Text of the last error on this handle ("" if none); valid until the next call on the handle. */
const char* ctr_last_error(const ctr_handle* h);

#ifdef __cplusplus
}
#endif
#endif /* CTR_H_ */

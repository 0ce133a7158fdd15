// Host-side internals of libctr: the handle and the launch helpers shared by the .cu files.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/ctr.h"

namespace ctr {

#define CTR_MAX_ARMIJO 32
#define CTR_STAT_SWEEPS 4096 /* ring capacity, in sweeps */
#define CTR_PROF_MAX 32768
#ifndef CTR_MAX_BASIS
#define CTR_MAX_BASIS 4 /* stored unit gradients b_0..b_3 used for re-orthogonalisation (S24); valid: 1..4 */
#endif
#define CTR_NCOUNTERS 8
#define CTR_REDUCE_BLOCKS 1184 /* grid cap of the grid-stride reduction kernels: 148 SMs x 8 */

// Plain-data description of the problem, passed by value to every kernel.
struct Dims {
  int ndim;
  int nx, ny, nz;
  int nviews, nu, nv;
  int c0x, c0y, c0z;      // grid line taken as coordinate origin (n/2)
  int npix;               // voxels per slice / volume
  int nray;               // rays per slice / volume
  int G, B, V;            // groups (of V slices), true batch, slices per group
  int GS, LQ;             // slice-interleaved layout: super-groups of LQ groups (LQ*V slices), G = GS*LQ
  int nvp;                // nviews padded to a multiple of 16 (row length of win2)
  float xlo, ylo, zlo;    // mm, lower corner of the grid
  float dx, dy, dz;       // mm
  float dso, dsd;
  float inv_du, inv_dv;   // 1/pitch
  float dvz;              // dv/dz (3D: detector row pitch in voxel heights)
  float boff_u, boff_v;   // (n-1)/2 - off : bin = coord/pitch + boff
  float rvox;             // half diagonal of a voxel, mm
  int det_type;
};

// Per-slice device scalars (arrays of length Bp = G*V).
struct Scal {
  double* gamma;   // ||P^T r||^2
  float* a;        // CGLS step
  float* beta;     // CGLS beta
  float* sigma2;   // sigma^2 of the current sweep
  double* e0;      // energy at the sweep start
  double* g2;      // ||g||^2
  int* kacc;       // accepted Armijo index or -1
  float* tacc;     // accepted step
  unsigned* sel_prefix;  // radix-select state
  unsigned* sel_rank;
  float* ginv;     // 1/||g|| of the newest CGLS gradient (0 when g = 0)
  float* coef;     // [CTR_MAX_BASIS][Bp] projections of g on the stored unit gradients
  float* eco;      // [CTR_MAX_BASIS][Bp] lazy phase of CGLS: the true direction is s = s_hat - sum_i eco_i b_i
  float* dco;      // [CTR_MAX_BASIS][Bp] lazy phase of CGLS: the true iterate is u = u_hat - sum_i dco_i b_i
  // fused sigma selection (ctr_tv.cu): candidate lists of the first radix pass
  int* pred;            // top-11-bit bin of sigma^2 found by the previous sweep (the prediction; < 0: none)
  unsigned* cand_cnt;   // entries appended to the slice's candidate list by the current first pass
  unsigned* ovf;        // a block's staging buffer overflowed: the list is incomplete
  int* hit;             // 1: the winning bin is covered by the list, passes 2 and 3 run on the list
  int* fhit;            // 1: the fast first pass (k_tv_scan1f) found the winning bin inside its three-bin window
  int* lastbin;         // bin of sigma^2 in the last sweep of the previous outer iteration (< 0: none)
  int* jump;            // by how many bins sigma^2 moved across the last Step 1 (CGLS): sigma^2 grows by 1.2-2 x there,
                        // i.e. 2-9 bins, smoothly from one outer iteration to the next, so the first sweep after CGLS
                        // predicts lastbin + jump instead of missing its candidate list every time
};

// stored system matrix, sliced ELL (ctr_ell.cuh)
struct EllTable {
  float2* tab;    // (index, weight) pairs
  int* cap;       // [warps] slabs per warp of 32 rows
  size_t* off;    // [warps] offset of the warp's slabs in tab
  size_t nrows, bytes;
};

// Ring of sweep records (ctr_get_stats). The slot of the CURRENT sweep is taken from a device-side sweep counter
// (advanced by k_tv_apply), not from a host value baked into the launch, so that a captured CUDA graph of one outer
// iteration writes consecutive records when it is replayed.
struct StatRing {
  ctr_sweep_stat* base;             // [CTR_STAT_SWEEPS][Bp]
  unsigned long long* sweep;        // device counter: sweeps finished since the last reset
  int Bp;
#ifdef __CUDACC__
  __device__ __forceinline__ ctr_sweep_stat* slot() const { return base + (size_t)(__ldcg(sweep) % CTR_STAT_SWEEPS) * Bp; }
#endif
};

struct TvParams {
  float lambda, eps, c_armijo;
  int kmax;
  int weights_mode;
  float t[CTR_MAX_ARMIJO];
};

}  // namespace ctr

namespace ctr {
// what a captured outer iteration has baked in (ctr_reconstruct)
struct GraphKey {
  const float* sino;
  float* img;
  ctr_params p;   // n_outer and warm_start zeroed
  unsigned long long sel_k;
};
}  // namespace ctr

struct ctr_handle {
  ctr_geometry g;
  ctr_params p;
  ctr::Dims d;
  int device;
  // geometry tables
  float4* rays;    // [nviews*nv*nu]  (2D: {x0, m, +-L, K}); 3D: see ctr_cone.cu
  float4* rays2;   // 3D second half of the ray record
  float2* views;   // [nviews] (cos, sin)
  double2* viewsd; // [nviews] (cos, sin) in fp64 (2D; Eq. (11) backprojector)
  unsigned short* win;  // [nviews][npix] first_bin << 4 | count (2D gather window table)
  unsigned short* win2; // same table as [npix][nvp] (views contiguous), slice-interleaved path only
  int win_ok;           // table usable (nu <= 4095 and every count <= 15)
  float* imgT;          // transposed copy of the image being projected, [G][nx][ny]
  // scratch, internal layout [G][n][V]
  size_t nimg, nsino;  // floats per internal image / sinogram (all groups)
  float *ximg, *bsino, *r, *q, *s, *gimg, *v, *w, *n0;
  int* qidx;            // [nquad][hits_cap] ray index * LQ (-1: padding): quad hit table of the batched gather P^T
  float4* qwts;         // [nquad][hits_cap] p_ij of that ray in the four pixels of the 2 x 2 quad
  int* qcnt;            // [nquad] entries used per quad
  int hits_cap;
  float2* rt_tab;       // stored P for batches: per ray (pixel index * LQ, p_ij), padded to chunks of 16 (ctr_si.cu)
  int* rt_cnt;          // [nray] entries per ray
  unsigned* rt_off;     // [nray] offset of the ray's entries in rt_tab
  size_t rt_bytes;
  ctr::EllTable ell_p, ell_pt;  // stored P (rows = rays) and P^T (rows = voxels), batch = 1 only; tab == NULL: on the fly
  int ell_p_blk;                // stored P indexes the blocked copy of its input (blk_index, ctr_fan_geom.cuh), kept in imgT
  unsigned* cand;       // [Bp][cand_cap] candidate lists (bit patterns of N0^2 near the predicted sigma^2)
  unsigned cand_cap;
  float* usi;           // CGLS iterate in the slice-interleaved layout (batch > 1)
  float* basis;         // [CTR_MAX_BASIS][nimg] unit CGLS gradients (S24), allocated in ctr_create
  float* pbasis;        // [CTR_MAX_BASIS][nsino] their projections P b_i (lazy phase of CGLS, ctr_api.cu)
  float* qprev;         // [nsino] P s of the previous CGLS iteration while the P b_i are being formed
  double* part2;        // block partials of the sinogram-side dot products <P b_i, r>
  int dots_blocks;      // resident blocks of k_reorth_dots on this device (its grid size)
  double* part;
  size_t part_len;
  unsigned* counters;   // [CTR_NCOUNTERS][G]
  unsigned* hist;       // [Bp][2048]
  ctr::Scal sc;
  void* scal_block;
  ctr_sweep_stat* stats;     // device ring [CTR_STAT_SWEEPS][Bp]
  unsigned long long* d_sweep;  // device copy of sweep_count (StatRing)
  long long sweep_count;     // sweeps recorded since the last reset
  unsigned long long sel_k;  // rank of the sigma order statistic (1-based), from the current quantile
  float sel_q;
  cudaStream_t last_stream;
  long long launches;
  // CUDA graph of the steady-state outer iteration (batch = 1)
  cudaStream_t gstream;       // capture stream (never executes anything)
  cudaGraphExec_t graph_exec;
  ctr::GraphKey graph_key;
  long long graph_launches;   // kernels per replay
  // optional event profiler (ctr_profile_*)
  int prof_on;
  int prof_n;                 // intervals recorded
  cudaEvent_t* prof_ev;       // [2 * CTR_PROF_MAX]
  unsigned char* prof_kind;   // [CTR_PROF_MAX]
  char err[256];
  char path_info[160];
};

namespace ctr {

inline int set_err(ctr_handle* h, int code, const char* msg) {
  if (h) snprintf(h->err, sizeof(h->err), "%s", msg);
  return code;
}

inline int cuda_fail(ctr_handle* h, cudaError_t e, const char* where) {
  if (h) snprintf(h->err, sizeof(h->err), "%s: %s", where, cudaGetErrorString(e));
  return CTR_ECUDA;
}

#define CTR_CUDA(h, call)                                         \
  do {                                                            \
    cudaError_t e__ = (call);                                     \
    if (e__ != cudaSuccess) return ctr::cuda_fail(h, e__, #call); \
  } while (0)

#define CTR_LAUNCHED(h)                                                       \
  do {                                                                        \
    (h)->launches++;                                                          \
    cudaError_t e__ = cudaPeekAtLastError();                                  \
    if (e__ != cudaSuccess) return ctr::cuda_fail(h, e__, "kernel launch");   \
  } while (0)

// RAII interval of the event profiler: records an event pair on `st` around a scope when enabled.
struct ProfScope {
  ctr_handle* h;
  cudaStream_t st;
  int slot;
  ProfScope(ctr_handle* h_, int kind, cudaStream_t st_) : h(h_), st(st_), slot(-1) {
    if (h->prof_on && h->prof_n < CTR_PROF_MAX) {
      slot = h->prof_n++;
      h->prof_kind[slot] = (unsigned char)kind;
      cudaEventRecord(h->prof_ev[2 * slot], st);
    }
  }
  ~ProfScope() {
    if (slot >= 0) cudaEventRecord(h->prof_ev[2 * slot + 1], st);
  }
};

// implemented in ctr_fan.cu (2D fan beam, V = 1 or 4)
int fan_build_tables(ctr_handle* h);
int fan_forward(ctr_handle* h, const float* img, float* out, int mode, const float* bs, cudaStream_t st);
int fan_back(ctr_handle* h, const float* sino, float* out, int mode, const float* s, float* u, cudaStream_t st);
int fan_back_eq11(ctr_handle* h, const float* sino, float* img, cudaStream_t st);  // ABI layouts, any batch
// implemented in ctr_si.cu (2D fan beam, batch > 1: slice-interleaved layout [n][LQ] of float4)
int si_forward(ctr_handle* h, const float* img, float* out, int mode, const float* bs, cudaStream_t st);
int si_back(ctr_handle* h, const float* sino, float* out, int mode, const float* s, float* u, cudaStream_t st);
int si_build_hits(ctr_handle* h);
int si_build_raytab(ctr_handle* h);
int si_from_abi(ctr_handle* h, const float* src, float* dst, size_t n, cudaStream_t st);   // [B][n] -> SI
int si_to_abi(ctr_handle* h, const float* src, float* dst, size_t n, cudaStream_t st);     // SI -> [B][n]
int si_from_planar(ctr_handle* h, const float* src, float* dst, size_t n, cudaStream_t st); // [G][n] float4 -> SI
int si_to_planar(ctr_handle* h, const float* src, float* dst, size_t n, cudaStream_t st);   // SI -> [G][n] float4
// implemented in ctr_cone.cu (3D cone beam, V = 1)
int cone_build_tables(ctr_handle* h);
int cone_forward(ctr_handle* h, const float* img, float* out, int mode, const float* bs, cudaStream_t st);
int cone_back(ctr_handle* h, const float* sino, float* out, int mode, const float* s, float* u, cudaStream_t st);
// implemented in ctr_tv.cu
int tv_update_weights(ctr_handle* h, const float* f, float* w, cudaStream_t st);
int tv_sweep(ctr_handle* h, float* f, const float* v, const float* w, float lambda, int clamp, cudaStream_t st);  // weights from the planes w
// weights + sweep, no planes; pos: bit 0 = first sweep after Step 1, bit 1 = last sweep of the outer iteration
int tv_sweep_fused(ctr_handle* h, float* f, const float* v, float lambda, int clamp, int pos, cudaStream_t st);
int tv_clamp(ctr_handle* h, float* f, cudaStream_t st);
// implemented in ctr_api.cu: finishing pass of a segmented reduction (block partials in h->part)
enum { CTR_FIN_ALPHA = 0, CTR_FIN_COEF = 1 };
int reduce_finish(ctr_handle* h, int mode, int N, int nblk, int i0, int nb, int first, cudaStream_t st);

}  // namespace ctr

// ptycho_kernels.cu — sm_100a kernels and the C ABI (include/ptycho.h) of the multislice ptychography hot path.
//
// Path, all on the caller's stream:
//   k_setup_prop     H5 tables  hx_i[qx], hy_i[qy] (separable Fresnel + tilt phases, fp64 math -> fp32)
//   setup_pos_one    H0 position split (fp32, reading R2) + H2 shift ramps rx_j, ry_j + bounds flag (R4)
//   k_probe_fft      H1 P~_k = F(P_k)
//   k_forward        H2..H6 one CTA per (position j, mode k): field in registers, 2S in-register 2-D FFTs,
//                    entering waves Psi_{i,k} stashed for the adjoint, far field psi~_k written out
//   k_loss           H7,H8 mode-summed intensity, per-pixel loss in fp64, detector weight w
//   k_backward       H9,H10,H12,H13 one CTA per (j,k): adjoint chain, per-(j,k,i) patch gradients,
//                    per-(j,k) probe-gradient spectra and position-gradient terms
//   k_backward_pair  the same for TWO modes per CTA (even mode counts): the idle mode's field and the first mode's
//                    patch gradient live in tensor memory (TMEM), only the pair's sum is staged
//   k_gather_object  H11 deterministic owner-computes scatter-add: every object pixel sums the patch
//                    gradients that cover it in fixed (j,k) order — no float atomics
//   k_gather_object_w the same with the windows split over the warps of a block (objects with few tiles: configs 1, 2)
//   k_single         S = 1: H2..H13 of one position in one persistent CTA, all modes in turn (configs 1, 2)
//   k_reduce_probe / k_probe_ifft / k_finalize   H12 tail, loss and position-gradient sums
//   k_step_object / k_step_probe   H14 LSQML-style step-size terms from what the backward pass staged (no second pass through
//                    the chain); k_alpha_pos / k_gather_willum / k_objtrans: the per-position-alpha weights and the probe-view
//                    preconditioner of LSQML; k_axpy / k_lsqml_* H15
//   regularizers.cuh cost / constraint regularisers and Adam
// The CPU oracle under oracle/ shares nothing with this file.
#include <cuda_runtime.h>
#include <math_constants.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#include <atomic>
#include <mutex>
#include <vector>

#include "../../include/ptycho.h"
#include "fft_core.cuh"

// Build units.  The file compiles either as one translation unit (PTK_ONLY_GEO undefined) or as four that the build compiles in
// parallel (ptycho.build): PTK_ONLY_GEO = 64 / 128 / 256 holds the chain kernels of that geometry and their launch sequences
// (run_forward / run_gradient), PTK_ONLY_GEO = 0 the C ABI, the geometry-independent kernels and regularizers.cuh.
#ifndef PTK_ONLY_GEO
#define PTK_ONLY_GEO -1
#endif
#define PTK_HAS_GEO(n) (PTK_ONLY_GEO == -1 || PTK_ONLY_GEO == (n))
#define PTK_HAS_ABI (PTK_ONLY_GEO <= 0)

using namespace ptk;

// per-thread launch counter and optional profiling record (ptycho_launch_count, ptycho_profile_*): shared by all build units
struct ProfMark { cudaEvent_t ev; int kind; };          // kind < 0: start-of-call marker
namespace ptk_state {
extern thread_local int64_t g_launches;
extern thread_local bool g_prof_on;
extern thread_local std::vector<ProfMark> g_prof;
#if PTK_HAS_ABI
thread_local int64_t g_launches = 0;
thread_local bool g_prof_on = false;
thread_local std::vector<ProfMark> g_prof;
#endif
}  // namespace ptk_state
using namespace ptk_state;

// launch sequences of one geometry (defined in that geometry's build unit); kp points at the caller's KP
struct GradArgs { pt_c64* gO; pt_c64* gP; float* gX; float* illum; const float* illum_prev; float* step_terms; double* loss; float* loss_per_pos;
                  const cudaEvent_t* chunk_ready; };
namespace ptk_geo {
int run_forward_64(const pt_problem* p, const void* kp, double* loss_d, float* loss_per_pos_d, float* model_intensity_d, cudaStream_t st);
int run_forward_128(const pt_problem* p, const void* kp, double* loss_d, float* loss_per_pos_d, float* model_intensity_d, cudaStream_t st);
int run_forward_256(const pt_problem* p, const void* kp, double* loss_d, float* loss_per_pos_d, float* model_intensity_d, cudaStream_t st);
int run_gradient_64(const pt_problem* p, const void* kp, const GradArgs* a, cudaStream_t st);
int run_gradient_128(const pt_problem* p, const void* kp, const GradArgs* a, cudaStream_t st);
int run_gradient_256(const pt_problem* p, const void* kp, const GradArgs* a, cudaStream_t st);
}  // namespace ptk_geo

namespace {

constexpr int kStatusOOB = 1, kStatusNonfinite = 2;
constexpr int kReduceZ = 8;          // k_reduce_probe: partial sums per chunk

// ------------------------------------------------------------------------------------------------
// workspace layout (host + device agree through this POD)
// ------------------------------------------------------------------------------------------------
struct Ws {
  int32_t* status;     // [16]
  cf* hx;              // [max(S-1,1)][N]   pre-scaled by 1/N^2
  cf* hy;              // [max(S-1,1)][N]
  cf* ramps;           // [J][2][N]  (rx, ry)
  int32_t* r0;         // [J][2]  (y, x)
  float* delta;        // [J][2]
  int32_t* rows;       // [J]     checked row of positions / intensity for each batch entry (k_setup_pos)
  cf* Pt;              // [M][N^2]  F-native, unscaled
  cf* Qt;              // [M][N^2]  F-native: F(dPhat_k) for the step-size sweep
  double2* gPt_acc;    // [M][N^2]  F-native accumulators
  double2* gPt_part;   // [kReduceZ][M][N^2]  partial sums of one chunk (k_reduce_probe)
  double* loss_pp;     // [J][CL]
  double* posg_part;   // [J][M][CL][2]
  double* step_oi;     // [J][S][6]       step-size sweep: (numO, denO) of slice i; bilinear mode also (numX_y, denX_y, numX_x, denX_x)
  double* step_pp;     // [J][M][CL][6]   step-size sweep: (numP, denP, numX_y, denX_y, numX_x, denX_x) of one mode (and rank)
  cf* dOhat;           // [S][ony][onx]      (step sizes only)
  float4* O2;          // [S][ony][onx]      the object with its partner: O2[y][x] = (O[y][x], O[y][x + D]), D = the distance of a thread's
                       //                    registers 2p, 2p + 1 in the patch (k_pair_object): one 16-byte copy brings both
  // chunked
  cf* psit;            // [Jc][M][N^2]  F-native
  float* wdet;         // [Jc][N^2]     F-native
  cf* stash;           // [Jc][M][S][N^2]  R-native
  // staged by the backward pass: per chunk, or per BATCH position when stage_all (step sizes) — the launch sequence then hands
  // the kernels pointers already advanced to the chunk's first position (stage_chunk), so kernels index all three by jl
  cf* gTpart;          // [Jc|J][M or M/2][S][N^2]  R-native (staged_planes)
  cf* Gpart;           // [Jc|J][M][N^2]     F-native
  float* psimax;       // [Jc][M][S][CL]   ePIE: max |Psi_{i,k}|^2 of each rank's block (PT_EPIE only)
  float* tmax;         // [Jc][S]          ePIE: max |O_i|^2 over the window
  float4* Tb;          // [Jc][S][N^2]     raster: bilinearly sampled patches, each with its partner D pixels to the right, as O2
                       //                  (PT_SHIFT_BILINEAR_OBJECT only)
  float* alpha_ji;     // [Jc][S]          per-position object step sizes alpha_{O,i,j} (PT_WANT_WEIGHTED_ILLUM only)
  float* ilpart;       // [Jc|J][M or M/2][S][N^2]  R-native |Psi_{i,k}|^2 written by the backward kernels (step sizes; PT_WANT_ILLUM with paired modes)
  int32_t stage_all;   // the three staged arrays hold the whole batch (the step-size sweep reads them after the last chunk)
  int32_t Jc;
  size_t total;
};

inline size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }
// Two modes per CTA in the backward pass (k_backward_pair: the pair's patch gradients are summed on chip and staged once)
// whenever the number of modes is even; the flag PT_NO_MODE_PAIRS forces one mode per CTA (a debugging switch).
inline bool use_pairs(const pt_problem* p) { return (p->n_modes % 2) == 0 && !(p->flags & PT_NO_MODE_PAIRS); }
inline size_t staged_planes(const pt_problem* p) { return use_pairs(p) ? p->n_modes / 2 : p->n_modes; }   // gT planes per position
inline size_t cluster_of(int n) { return n == 256 ? 4 : 1; }   // CTAs per field (Geo<n>::CL)

// fixed bytes, bytes per position in flight (chunk), bytes per position of what the backward pass stages (patch gradients,
// probe partials), and the optional |Psi|^2 staging (illumination map with paired modes; mandatory for the step-size sweep)
struct WsSizes { size_t fixed, per_chunk, per_staged, per_il; bool il_needed; };
WsSizes ws_sizes(const pt_problem* p) {
  const size_t N = p->n, NN = N * N, M = p->n_modes, S = p->n_slices, J = p->n_batch, CL = cluster_of(p->n);
  const bool steps = (p->flags & PT_WANT_STEP_SIZES) != 0;
  size_t f = 256;
  f += 2 * align_up((S > 1 ? S - 1 : 1) * N * sizeof(cf));
  f += align_up(J * 2 * N * sizeof(cf)) + align_up(J * 2 * sizeof(int32_t)) + align_up(J * 2 * sizeof(float)) + align_up(J * sizeof(int32_t));
  f += 2 * align_up(M * NN * sizeof(cf)) + (1 + kReduceZ) * align_up(M * NN * sizeof(double2));       // gPt_acc + partial planes
  f += align_up(J * CL * sizeof(double)) + align_up(J * M * CL * 2 * sizeof(double));
  f += align_up(J * S * 6 * sizeof(double)) + align_up(J * M * CL * 6 * sizeof(double));
  if (steps) f += align_up(S * (size_t)p->obj_ny * p->obj_nx * sizeof(cf));
  f += align_up(S * (size_t)p->obj_ny * p->obj_nx * sizeof(float4));
  WsSizes z;
  z.fixed = f + 13 * 256;   // slack for the per-array alignment of the chunked part
  const size_t stash_el = (p->flags & PT_STASH_FP16) ? sizeof(cf) / 2 : sizeof(cf);   // binary16 pairs: 4 bytes per complex
  z.per_chunk = M * NN * sizeof(cf) + NN * sizeof(float) + M * S * NN * stash_el;
  if (steps) z.per_chunk += S * sizeof(float);
  if (p->shift_mode == PT_SHIFT_BILINEAR_OBJECT) z.per_chunk += S * NN * sizeof(float4);
  if (p->flags & PT_EPIE) z.per_chunk += (M * CL + 1) * S * sizeof(float) + 64;
  z.per_staged = staged_planes(p) * S * NN * sizeof(cf) + M * NN * sizeof(cf);
  z.il_needed = steps;
  z.per_il = 0;
  if (!(p->flags & PT_EPIE) && (steps || ((p->flags & PT_WANT_ILLUM) && use_pairs(p)))) z.per_il = staged_planes(p) * S * NN * sizeof(float);
  return z;
}
// Positions in flight for a workspace of `bytes`.  Without step sizes everything is per chunk; the optional |Psi|^2 staging is
// used when the whole batch still fits with it, or when the batch is chunked anyway, not when it alone would force chunking (a
// caller who sized the workspace for the batch without PT_WANT_ILLUM gets the same single chunk as before).  With step sizes
// the staged arrays are kept for the WHOLE batch when the workspace allows (stage_all): the sweep then reads them after the last
// chunk; otherwise each chunk is recomputed for the sweep.
struct ChunkPlan { size_t jc; bool il; bool stage_all; };
ChunkPlan plan_chunks(const pt_problem* p, size_t bytes) {
  const WsSizes z = ws_sizes(p);
  ChunkPlan c = {0, false, false};
  const size_t J = (size_t)p->n_batch;
  if (z.il_needed) {
    const size_t pp = z.per_chunk + z.per_staged + z.per_il;
    if (bytes < z.fixed + pp) return c;
    c.il = true;
    c.jc = (bytes - z.fixed) / pp;
    if (c.jc >= J) { c.jc = J; return c; }
    const size_t staged = J * (z.per_staged + z.per_il), floor_jc = J < 64 ? J : 64;
    if (bytes >= z.fixed + staged + floor_jc * z.per_chunk) {
      c.stage_all = true;
      c.jc = (bytes - z.fixed - staged) / z.per_chunk;
      if (c.jc > J) c.jc = J;
    }
    return c;
  }
  const size_t pp = z.per_chunk + z.per_staged;
  if (bytes < z.fixed + pp) return c;
  size_t jc0 = (bytes - z.fixed) / pp;
  if (jc0 > J) jc0 = J;
  c.jc = jc0;
  if (z.per_il) {
    size_t jc1 = (bytes - z.fixed) / (pp + z.per_il);
    if (jc1 > J) jc1 = J;
    if (jc1 >= 1 && (jc1 == J || jc0 < J)) { c.jc = jc1; c.il = true; }
  }
  return c;
}

int ws_layout(const pt_problem* p, void* base, size_t bytes, Ws* w) {
  const ChunkPlan plan = plan_chunks(p, bytes);
  if (plan.jc == 0) return PT_ERR_WORKSPACE;
  const size_t jc = plan.jc;
  const size_t N = p->n, NN = N * N, M = p->n_modes, S = p->n_slices, J = p->n_batch, CL = cluster_of(p->n);
  const size_t js = plan.stage_all ? J : jc;                       // positions the staged arrays hold
  const bool steps = (p->flags & PT_WANT_STEP_SIZES) != 0;
  char* c = (char*)base;
  size_t off = 0;
  auto take = [&](size_t n) { char* r = c + off; off += align_up(n); return (void*)r; };
  w->status = (int32_t*)take(256);
  w->hx = (cf*)take((S > 1 ? S - 1 : 1) * N * sizeof(cf));
  w->hy = (cf*)take((S > 1 ? S - 1 : 1) * N * sizeof(cf));
  w->ramps = (cf*)take(J * 2 * N * sizeof(cf));
  w->r0 = (int32_t*)take(J * 2 * sizeof(int32_t));
  w->delta = (float*)take(J * 2 * sizeof(float));
  w->rows = (int32_t*)take(J * sizeof(int32_t));
  w->Pt = (cf*)take(M * NN * sizeof(cf));
  w->Qt = (cf*)take(M * NN * sizeof(cf));
  w->gPt_acc = (double2*)take(M * NN * sizeof(double2));
  w->gPt_part = (double2*)take(kReduceZ * M * NN * sizeof(double2));
  w->loss_pp = (double*)take(J * CL * sizeof(double));
  w->posg_part = (double*)take(J * M * CL * 2 * sizeof(double));
  w->step_oi = (double*)take(J * S * 6 * sizeof(double));
  w->step_pp = (double*)take(J * M * CL * 6 * sizeof(double));
  w->dOhat = steps ? (cf*)take(S * (size_t)p->obj_ny * p->obj_nx * sizeof(cf)) : nullptr;
  w->O2 = (float4*)take(S * (size_t)p->obj_ny * p->obj_nx * sizeof(float4));
  w->psit = (cf*)take(jc * M * NN * sizeof(cf));
  w->wdet = (float*)take(jc * NN * sizeof(float));
  w->stash = (cf*)take(jc * M * S * NN * ((p->flags & PT_STASH_FP16) ? sizeof(cf) / 2 : sizeof(cf)));
  w->gTpart = (cf*)take(js * staged_planes(p) * S * NN * sizeof(cf));
  w->Gpart = (cf*)take(js * M * NN * sizeof(cf));
  w->psimax = (p->flags & PT_EPIE) ? (float*)take(jc * M * S * CL * sizeof(float)) : nullptr;
  w->tmax = (p->flags & PT_EPIE) ? (float*)take(jc * S * sizeof(float)) : nullptr;
  w->Tb = p->shift_mode == PT_SHIFT_BILINEAR_OBJECT ? (float4*)take(jc * S * NN * sizeof(float4)) : nullptr;
  w->alpha_ji = steps ? (float*)take(jc * S * sizeof(float)) : nullptr;
  w->ilpart = plan.il ? (float*)take(js * staged_planes(p) * S * NN * sizeof(float)) : nullptr;
  w->stage_all = plan.stage_all ? 1 : 0;
  w->Jc = (int32_t)jc;
  w->total = off;
  return off <= bytes ? PT_OK : PT_ERR_WORKSPACE;
}

// ------------------------------------------------------------------------------------------------
// kernel parameter block
// ------------------------------------------------------------------------------------------------
struct KP {
  int N, M, S, ony, onx, J;          // J = batch size
  int Jtot;                          // rows of positions / intensity (n_pos_total)
  int Mg;                            // patch-gradient planes per position in the staging buffer: M, or M/2 after k_backward_pair
  int Mi;                            // |Psi|^2 planes per position in the staging buffer: M, or M/2 after k_backward_pair (the pair's sum)
  int j0, jc;                        // current chunk: batch-local offset and count
  float chi_scale;                   // step-size sweep: chi = -chi_scale gPhi (1; 2 under PT_LSQML_MODULUS_CHI, reading R31)
  float px, bandlim2;                // bandlim2 = (0.5*bandlimit*N)^2 or < 0 when off
  int loss; float loss_c, eps;
  int bilinear;                      // PT_SHIFT_BILINEAR_OBJECT: probe unshifted, patches sampled with four taps (reading R1)
  const cf* object; const cf* probe; const float* positions; const float* intensity; const int32_t* batch_idx;
  Ws w;
};

__device__ __forceinline__ int signed_freq(int q, int N) { return q < N / 2 ? q : q - N; }

// ------------------------------------------------------------------------------------------------
// H5 tables: hx_i[q] = exp(-i pi lambda dz kx^2 + 2 pi i dz kx tan(tx)) / N^2, hy_i likewise without the scale
// (readings R7, R8).  fp64 math, one thread per (i, axis, q).
// ------------------------------------------------------------------------------------------------
struct PropArgs { int N, nprop; double px, lambda, tx, ty; cf* hx; cf* hy; float dz[64]; int i0; };
__global__ void k_setup_prop(PropArgs a) {
  int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= a.nprop * 2 * a.N) return;
  int q = idx % a.N, axis = (idx / a.N) & 1, il = idx / (2 * a.N);
  double dz = (double)a.dz[il];
  double k = (double)signed_freq(q, a.N) / (double)a.N / a.px;
  double t = axis == 0 ? tan(a.tx * 1e-3) : tan(a.ty * 1e-3);
  double ang = -CUDART_PI * a.lambda * dz * k * k + 2.0 * CUDART_PI * dz * k * t;
  double s, c;
  sincos(ang, &s, &c);
  if (axis == 0) {
    double sc = 1.0 / ((double)a.N * (double)a.N);
    a.hx[(size_t)(a.i0 + il) * a.N + q] = make_float2((float)(c * sc), (float)(s * sc));
  } else {
    a.hy[(size_t)(a.i0 + il) * a.N + q] = make_float2((float)c, (float)s);
  }
}

// ------------------------------------------------------------------------------------------------
// H0 + H2 tables: position split in fp32 exactly as the reading R2 states it (no FMA contraction), bounds
// flag (R4: clamp + raise), shift ramps rx[q] = exp(-2 pi i f(q) dx), ry likewise.
// N threads per position (thread q writes the ramps' entry q); launched inside k_pair_object's grid (below).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void setup_pos_one(const KP& P, int jb, int q) {
  const int N = P.N;
  int row = P.batch_idx ? P.batch_idx[jb] : jb;
  if (row < 0 || row >= P.Jtot) {                                 // a batch entry outside the tables: clamp + raise, as R4
    if (q == 0) atomicOr(P.w.status, kStatusOOB);
    row = row < 0 ? 0 : P.Jtot - 1;
  }
  if (q == 0) P.w.rows[jb] = row;                                 // k_loss reads the checked row
  float d[2]; int r0[2];
#pragma unroll
  for (int a = 0; a < 2; ++a) {
    float X = P.positions[2 * row + a];
    float p = __fdiv_rn(X, P.px);
    float c = __fsub_rn(p, (float)(N / 2));
    float fl = floorf(P.bilinear ? c : __fadd_rn(c, 0.5f));    // bilinear mode: i0 = floor(c), f = c - i0 in [0, 1)
    d[a] = __fsub_rn(c, fl);
    int r = (int)fl;
    int lim = (a == 0 ? P.ony : P.onx) - N - (P.bilinear ? 1 : 0);   // bilinear taps reach i0 + N
    if (r < 0 || r > lim) {
      if (q == 0) atomicOr(P.w.status, kStatusOOB);
      r = r < 0 ? 0 : lim;
    }
    r0[a] = r;
  }
  if (q == 0) {
    P.w.r0[2 * jb] = r0[0]; P.w.r0[2 * jb + 1] = r0[1];
    P.w.delta[2 * jb] = d[0]; P.w.delta[2 * jb + 1] = d[1];
  }
  const float f = (float)signed_freq(q, N) / (float)N;
  float s, c;
  const float dsx = P.bilinear ? 0.f : d[1], dsy = P.bilinear ? 0.f : d[0];   // bilinear mode: the probe is not shifted (R = 1)
  sincospif(-2.0f * f * dsx, &s, &c);
  P.w.ramps[((size_t)jb * 2 + 0) * N + q] = make_float2(c, s);     // rx
  sincospif(-2.0f * f * dsy, &s, &c);
  P.w.ramps[((size_t)jb * 2 + 1) * N + q] = make_float2(c, s);     // ry
}

// O2[y][x] = (O[y][x], O[y][x + D]) for every slice (zero where x + D leaves the row: no window reads those as a first element)
// The same launch clears up to three arrays of the gradient call (probe-gradient accumulator, grad_object, illumination map): a
// small problem's step is a dozen launches of a few microseconds each, every launch saved counts.
// Blocks [nb_obj, gridDim.x) do the position set-up (k_setup_pos of earlier builds: 256 / N positions per block) — one launch for the
// whole prologue besides the probe transform and the propagator tables.
__global__ void __launch_bounds__(256) k_pair_object(KP P, int D, float* za, size_t na, float* zb, size_t nb, float* zc, size_t nc, unsigned nb_obj) {
  if (blockIdx.x >= nb_obj) {
    const int jb = (int)(blockIdx.x - nb_obj) * (256 / P.N) + (int)threadIdx.x / P.N;
    if (jb < P.J) setup_pos_one(P, jb, (int)threadIdx.x % P.N);
    return;
  }
  const size_t n = (size_t)P.S * P.ony * P.onx, i = (size_t)blockIdx.x * blockDim.x + threadIdx.x, stride = (size_t)nb_obj * blockDim.x;
  for (size_t j = i; j < na; j += stride) za[j] = 0.f;
  for (size_t j = i; j < nb; j += stride) zb[j] = 0.f;
  for (size_t j = i; j < nc; j += stride) zc[j] = 0.f;
  if (i >= n) return;
  const int x = (int)(i % P.onx);
  const cf a = P.object[i], b = x + D < P.onx ? P.object[i + D] : make_float2(0.f, 0.f);
  P.w.O2[i] = make_float4(a.x, a.y, b.x, b.y);
}

// ------------------------------------------------------------------------------------------------
// block-wide deterministic sum of NV doubles per thread; result valid in thread 0
// ------------------------------------------------------------------------------------------------
template <int T, int NV>
__device__ __forceinline__ void block_sum(double (&val)[NV], double* red /* [T/32][NV] */) {
#pragma unroll
  for (int i = 0; i < NV; ++i)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) val[i] += __shfl_xor_sync(0xffffffffu, val[i], o);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0)
#pragma unroll
    for (int i = 0; i < NV; ++i) red[w * NV + i] = val[i];
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      double s = 0.0;
      for (int ww = 0; ww < T / 32; ++ww) s += red[ww * NV + i];
      val[i] = s;
    }
  }
  __syncthreads();
}

template <class G> constexpr int min_blocks() { return G::T == 512 ? 1 : 4; }

// ------------------------------------------------------------------------------------------------
// Shared memory of the FFT kernels:
//   [ exchange buffer XBUF | twiddles TW | cluster twiddles TW2 (CL = 4 only) | reduction scratch 1 KB |
//     chain kernels only: hy tables 2 x NF | prefetch slots PF16 x T x 16 B ]
// Global data a slice needs (object patch T_i, stashed wave Psi_i) is brought in with cp.async into slots that
// belong to the thread that will consume them, so no barrier or mbarrier is involved: "early" slots (the PF16
// region) are filled one whole FFT pair ahead, "late" slots live in the calling warp's own X1 exchange region,
// which is idle between the end of fft2_inv_head and the next fft2_fwd (16 slots of 16 B per lane).
// ------------------------------------------------------------------------------------------------
template <class G> constexpr size_t fft_smem_bytes() { return (size_t)(Lay<G>::XBUF + Lay<G>::TW + (G::CL > 1 ? G::N : 0)) * sizeof(cf) + 1024; }
template <class G> constexpr size_t chain_smem_bytes() { return fft_smem_bytes<G>() + (size_t)(G::HXS ? 4 : 2) * G::NF * sizeof(cf) + (size_t)G::PF16 * G::T * 16; }
template <class G>
struct ChainSmem {
  cf* sm; cf* tw; cf* tw2; double* red; cf* hyS; cf* hxS; float4* pf; float4* xs;
  __device__ __forceinline__ ChainSmem(unsigned char* raw, int t) {
    typedef Lay<G> L;
    sm = (cf*)raw; tw = sm + L::XBUF; tw2 = tw + L::TW; red = (double*)(tw2 + (G::CL > 1 ? G::N : 0));
    hyS = (cf*)((unsigned char*)red + 1024);                            // hy tables of two consecutive propagations, then hx likewise
    hxS = hyS + 2 * G::NF;                                              // (G::HXS only; else the early slots start here)
    pf = (float4*)(hxS + (G::HXS ? 2 : 0) * G::NF) + t;                                // early 16-byte slot s: pf[s * T]
    xs = (float4*)(sm + (t >> 5) * L::X1_WARP) + (t & 31);              // late 16-byte slot s:  xs[s * 32]
  }
  // twiddle tables; the caller synchronises the CTA before the first transform
  __device__ __forceinline__ void fill_tables(int t) {
    for (int i = t; i < Lay<G>::TW; i += G::T) Lay<G>::fill_twiddle(tw, i);
    for (int i = t; i < (G::CL > 1 ? G::N : 0); i += G::T) FL<G>::fill_tw2(tw2, i);
  }
};
__device__ __forceinline__ void cp_async16(void* dst_smem, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
// every thread asks for the 128-byte line at p to be brought into L2 (fire and forget)
__device__ __forceinline__ void l2_prefetch_line(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ void cp_async8(void* dst_smem, const void* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
// reduced-precision stash (PT_STASH_FP16): four complex64 <-> eight binary16 in one 16-byte word, round to nearest even
__device__ __forceinline__ uint32_t pack_h2(float a, float b) {
  uint32_t r; asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(b), "f"(a)); return r;     // low half = a
}
__device__ __forceinline__ cf unpack_h2(uint32_t u) {
  float lo, hi;
  asm("{.reg .f16 l, h; mov.b32 {l, h}, %2; cvt.f32.f16 %0, l; cvt.f32.f16 %1, h;}" : "=f"(lo), "=f"(hi) : "r"(u));
  return make_float2(lo, hi);
}
// 16-byte read-only load pinned where it is written (asm volatile keeps its place among the other memory operations)
__device__ __forceinline__ float4 ld_nc16(const float4* p) {
  float4 v;
  asm volatile("ld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
  return v;
}
// one-instruction bulk copy global -> shared with completion on an mbarrier (the TMA engine moves the bytes)
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void bulk_load(void* dst_smem, const void* src, unsigned bytes, uint64_t* bar) {
  const unsigned b = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(b), "r"(bytes) : "memory");
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"((unsigned)__cvta_generic_to_shared(dst_smem)),
               "l"(src), "r"(bytes), "r"(b) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  const unsigned b = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile("{\n.reg .pred p;\nWAIT_%=:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@!p bra WAIT_%=;\n}" ::"r"(b), "r"(parity) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
// ------------------------------------------------------------------------------------------------
// H1: P~_k = F(P_k), stored Fourier-native.  Also used for Q~_k = F(dPhat_k) with a scale (step-size sweep, O14:
// in = raster grad_probe, scale = -1 / (delta_p + 1)).  One CTA (CL = 4: one cluster) per mode.
// ------------------------------------------------------------------------------------------------
template <class G>
__global__ void __launch_bounds__(G::T, min_blocks<G>()) k_probe_fft(const cf* in, cf* out, float scale, const float* precond, float delta_p) {
  typedef Lay<G> L; typedef FL<G> F;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int t = threadIdx.x, k = blockIdx.x / G::CL;
  const unsigned rk = Fft<G>::rank();
  ChainSmem<G> cs(smem_raw, t);
  cs.fill_tables(t);
  __syncthreads();
  cf v[32];
  const cf* src = in + (size_t)k * F::NNF;
#pragma unroll
  for (int r = 0; r < 32; ++r) {
    const int pix = F::pix_y(rk, t, r) * F::NF + F::pix_x(rk, t, r);
    // step-size sweep with the probe-view preconditioner (R25): dPhat = -gP / (precond + delta_p)
    v[r] = cscale(src[pix], precond ? -1.0f / (precond[pix] + delta_p) : scale);
  }
  Fft<G>::fwd(v, cs.sm, cs.tw, cs.tw2, t, rk);
  cf* dst = out + ((size_t)k * G::CL + rk) * F::NNS;
#pragma unroll
  for (int r = 0; r < 32; ++r) dst[L::native(t, r)] = v[r];
  Fft<G>::end_fourier();
}

// H12 tail: gP_k = Finv(gP~_k): Fourier-native double accumulators -> raster complex64 (overwrite or add)
template <class G>
__global__ void __launch_bounds__(G::T, min_blocks<G>()) k_probe_ifft(const double2* acc, cf* out, int accumulate, double extra_scale) {
  typedef Lay<G> L; typedef FL<G> F;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int t = threadIdx.x, k = blockIdx.x / G::CL;
  const unsigned rk = Fft<G>::rank();
  ChainSmem<G> cs(smem_raw, t);
  cs.fill_tables(t);
  Fft<G>::begin_fourier();
  __syncthreads();
  cf v[32];
  const double sc = extra_scale / ((double)F::NF * (double)F::NF);
  const double2* a0 = acc + ((size_t)k * G::CL + rk) * F::NNS;
#pragma unroll
  for (int r = 0; r < 32; ++r) { double2 a = a0[L::native(t, r)]; v[r] = make_float2((float)(a.x * sc), (float)(a.y * sc)); }
  Fft<G>::inv(v, cs.sm, cs.tw, cs.tw2, t, rk);
  cf* dst = out + (size_t)k * F::NNF;
#pragma unroll
  for (int r = 0; r < 32; ++r) {
    cf* d = dst + F::pix_y(rk, t, r) * F::NF + F::pix_x(rk, t, r);
    if (accumulate) { cf o = *d; *d = make_float2(o.x + v[r].x, o.y + v[r].y); } else *d = v[r];
  }
}

// ------------------------------------------------------------------------------------------------
// pointwise helpers on the register field
// ------------------------------------------------------------------------------------------------
// object patch pointer for (slice i, position window r0)
__device__ __forceinline__ const cf* patch_ptr(const KP& P, int i, int r0y, int r0x) {
  return P.object + ((size_t)i * P.ony + r0y) * P.onx + r0x;
}

// the thread's NXV values of an x-table (hx row or shift ramp rx), optionally scaled
template <class G>
__device__ __forceinline__ void load_xv(cf (&wxv)[FL<G>::NXV], const cf* row, int t, float scale) {
#pragma unroll
  for (int c = 0; c < FL<G>::NXV; ++c) wxv[c] = cscale(row[Lay<G>::f_qx(t, 0) + c * G::N], scale);
}

// v *= hx[qx] * hy[qy] (optionally conjugated) with the sharp band-limit mask (reading R9); hy from shared memory.
// Which of the thread's 32 Fourier pixels lie inside the band does not change from slice to slice: band_mask is formed once
// per kernel (bit r = register r is inside), the mask test is a bit test, and the branch on "mask on / off" is block-uniform
// and hoisted out of the unrolled loop (the five configs run with the mask off).
template <class G>
__device__ __forceinline__ uint32_t band_mask(float bandlim2, int t, unsigned rk) {
  typedef FL<G> F;
  uint32_t m = 0xffffffffu;
  if (bandlim2 >= 0.0f) {
    m = 0u;
#pragma unroll
    for (int r = 0; r < 32; ++r) {
      const int sx = signed_freq(F::fq_x(rk, t, r), F::NF), sy = signed_freq(F::fq_y(rk, t, r), F::NF);
      if (!((float)(sx * sx + sy * sy) > bandlim2)) m |= 1u << r;
    }
  }
  return m;
}
template <class G, bool CONJ, bool MASK>
__device__ __forceinline__ void apply_prop_body(cf (&v)[32], const cf (&wxv)[FL<G>::NXV], const cf* hyS, uint32_t inside, int t, unsigned rk) {
  typedef FL<G> F;
#pragma unroll
  for (int r = 0; r < 32; ++r) {
    const int qy = F::fq_y(rk, t, r);
    cf wx = wxv[F::fq_xsel(r)], wy = hyS[qy];
    if (CONJ) { wx.y = -wx.y; wy.y = -wy.y; }
    cf h = cmul(wx, wy);
    if (MASK && !((inside >> r) & 1u)) h = make_float2(0.f, 0.f);
    v[r] = cmul(v[r], h);
  }
}
template <class G, bool CONJ>
__device__ __forceinline__ void apply_prop_s(cf (&v)[32], const cf* hxrow, const cf* hyS, float bandlim2, uint32_t inside, int t, unsigned rk) {
  cf wxv[FL<G>::NXV];
  load_xv<G>(wxv, hxrow, t, 1.0f);
  if (bandlim2 >= 0.0f) apply_prop_body<G, CONJ, true>(v, wxv, hyS, inside, t, rk);
  else apply_prop_body<G, CONJ, false>(v, wxv, hyS, inside, t, rk);
}

// The backward kernels keep the mask test inside the loop: one more register live across their slice loop costs them more
// (spills: 57.5 -> 59.5 ms per step at config 3) than the test costs in the band-limited variant.
template <class G, bool CONJ, bool MASK>
__device__ __forceinline__ void apply_prop_body_t(cf (&v)[32], const cf (&wxv)[FL<G>::NXV], const cf* hyS, float bandlim2, int t, unsigned rk) {
  typedef FL<G> F;
#pragma unroll
  for (int r = 0; r < 32; ++r) {
    const int qy = F::fq_y(rk, t, r);
    cf wx = wxv[F::fq_xsel(r)], wy = hyS[qy];
    if (CONJ) { wx.y = -wx.y; wy.y = -wy.y; }
    cf h = cmul(wx, wy);
    if (MASK) {
      const int sx = signed_freq(F::fq_x(rk, t, r), F::NF), sy = signed_freq(qy, F::NF);
      if ((float)(sx * sx + sy * sy) > bandlim2) h = make_float2(0.f, 0.f);
    }
    v[r] = cmul(v[r], h);
  }
}
template <class G, bool CONJ>
__device__ __forceinline__ void apply_prop_t(cf (&v)[32], const cf* hxrow, const cf* hyS, float bandlim2, int t, unsigned rk) {
  cf wxv[FL<G>::NXV];
  load_xv<G>(wxv, hxrow, t, 1.0f);
  if (bandlim2 >= 0.0f) apply_prop_body_t<G, CONJ, true>(v, wxv, hyS, bandlim2, t, rk);
  else apply_prop_body_t<G, CONJ, false>(v, wxv, hyS, bandlim2, t, rk);
}

// ------------------------------------------------------------------------------------------------
// H2..H6 forward: one CTA (CL = 4: one cluster of four) per (j,k) pair of the chunk
// ------------------------------------------------------------------------------------------------
template <class G, int STASH>   // 0: nothing stashed (forward only); 1: Psi_i stashed as complex64; 2: as binary16 pairs (PT_STASH_FP16)
__global__ void __launch_bounds__(G::T, min_blocks<G>()) k_forward(KP P) {
  typedef Lay<G> L; typedef FL<G> F;
  constexpr int NF = F::NF, NNS = F::NNS, T = G::T, E = G::PF16, CL = G::CL;     // E pair slots early, 16 - E late
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int t = threadIdx.x;
  const unsigned rk = Fft<G>::rank();
  ChainSmem<G> cs(smem_raw, t);
  cf* sm = cs.sm; cf* tw = cs.tw;
  cs.fill_tables(t);
  Fft<G>::begin_fourier();
  const int pair = blockIdx.x / CL, jl = pair / P.M, k = pair - jl * P.M, jb = P.j0 + jl;
  const int r0y = P.w.r0[2 * jb], r0x = P.w.r0[2 * jb + 1];
  // patch source: the object window itself, or (bilinear mode) this position's resampled patches [S][NF][NF]
  const int S = P.S, onx = P.bilinear ? NF : P.onx;
  const size_t slice = P.bilinear ? (size_t)F::NNF : (size_t)P.ony * P.onx;
  const float4* ob2 = (P.bilinear ? P.w.Tb + (size_t)jl * S * F::NNF : P.w.O2 + ((size_t)r0y * P.onx + r0x)) +
                      (size_t)F::pix_y(rk, t, 0) * onx + F::pix_x(rk, t, 0);   // this thread's first pixel (with its partner), slice 0
  // H3 prefetch: patch values of register pairs [0, E) one FFT pair ahead into the thread's early slots
  auto early = [&](int i) {
    const float4* o2 = ob2 + (size_t)i * slice;
#pragma unroll
    for (int p = 0; p < E; ++p) cp_async16(cs.pf + p * T, o2 + F::patch_off(2 * p, onx));
    if (i < S - 1 && t < NF) {                                    // both tables of the propagation that ends iteration i (hx from global
      cp_async8(cs.hyS + (i & 1) * NF + t, P.w.hy + (size_t)i * NF + t);   // memory at its point of use exposed an L2 round trip per slice)
      if (G::HXS) cp_async8(cs.hxS + (i & 1) * NF + t, P.w.hx + (size_t)i * NF + t);
    }
    cp_async_commit();
  };
  early(0);
  __syncthreads();                                               // twiddle tables ready
  const cf* rx = P.w.ramps + (size_t)jb * 2 * NF;
  const cf* ry = rx + NF;
  cf v[32];
  {   // H2: R .* P~_k / N^2   (Fourier layout)
    const float4* pt = (const float4*)(P.w.Pt + ((size_t)k * CL + rk) * NNS);
    cf wxv[F::NXV];
    load_xv<G>(wxv, rx, t, 1.0f / (float)F::NNF);
#pragma unroll
    for (int p = 0; p < 16; ++p) {
      const float4 q = pt[p * T + t];
      v[2 * p] = cmul(make_float2(q.x, q.y), cmul(wxv[F::fq_xsel(2 * p)], ry[F::fq_y(rk, t, 2 * p)]));
      v[2 * p + 1] = cmul(make_float2(q.z, q.w), cmul(wxv[F::fq_xsel(2 * p + 1)], ry[F::fq_y(rk, t, 2 * p + 1)]));
    }
  }
  const uint32_t inside = band_mask<G>(P.bandlim2, t, rk);
  for (int i = 0; i < S; ++i) {
    Fft<G>::inv_head(v, sm, cs.tw2, t, rk);
    {   // registers [2E, 32) of T_i into the warp's idle X1 region
      const float4* o2 = ob2 + (size_t)i * slice;
#pragma unroll
      for (int p = E; p < 16; ++p) cp_async16(cs.xs + (p - E) * 32, o2 + F::patch_off(2 * p, onx));
      cp_async_commit();
    }
    L::phase1_inv(v, tw, t);                                     // Psi_{i,k}  (R-layout)
    cp_async_wait_all();
    float4* st = (float4*)(P.w.stash + (((size_t)pair * S + i) * CL + rk) * (STASH == 2 ? NNS / 2 : NNS));
    float hprev0 = 0.f, hprev1 = 0.f;                            // STASH == 2: the halves of the even pair, until the odd pair joins them
#pragma unroll
    for (int p = 0; p < 16; ++p) {                               // stash Psi_i ; H3+H4: Phi = Psi .* T_i
      if (STASH == 1) __stcs(st + p * T + t, make_float4(v[2 * p].x, v[2 * p].y, v[2 * p + 1].x, v[2 * p + 1].y));
      if (STASH == 2) {                                          // registers 2p-2 .. 2p+1 -> one 16-byte word of eight halves
        const float h0 = __uint_as_float(pack_h2(v[2 * p].x, v[2 * p].y)), h1 = __uint_as_float(pack_h2(v[2 * p + 1].x, v[2 * p + 1].y));
        if (p & 1) __stcs(st + (p >> 1) * T + t, make_float4(hprev0, hprev1, h0, h1));
        else { hprev0 = h0; hprev1 = h1; }
      }
      const float4 tt = p < E ? cs.pf[p * T] : cs.xs[(p - E) * 32];   // (T[2p], T[2p+1]): one 16-byte slot (k_pair_object)
      const cf T0 = make_float2(tt.x, tt.y), T1 = make_float2(tt.z, tt.w);
      v[2 * p] = cmul(v[2 * p], T0);
      v[2 * p + 1] = cmul(v[2 * p + 1], T1);
      if ((p & 3) == 3) L::phase1_fwd_row(v, p >> 2);            // registers [8 (p/4), 8 (p/4) + 8) are final: their row transform now,
                                                                 // between the bursts of stash stores (forward 46.4 -> 46.0 ms per step)
    }
    if (i + 1 < S) early(i + 1);
    Fft<G>::fwd_after_rows(v, sm, tw, cs.tw2, t, rk);            // F(Phi)    (Fourier layout)
    if (i < S - 1) apply_prop_s<G, false>(v, G::HXS ? cs.hxS + (i & 1) * NF : P.w.hx + (size_t)i * NF, cs.hyS + (i & 1) * NF, P.bandlim2, inside, t, rk);   // H5
  }
  float4* out = (float4*)(P.w.psit + ((size_t)pair * CL + rk) * NNS);   // H6: psi~ = F(Phi_{S-1}) / N
  const float sc = 1.0f / (float)NF;
#pragma unroll
  for (int p = 0; p < 16; ++p) out[p * T + t] = make_float4(v[2 * p].x * sc, v[2 * p].y * sc, v[2 * p + 1].x * sc, v[2 * p + 1].y * sc);
  Fft<G>::end_fourier();
}

// fp64 square root and reciprocal from a float32 seed and Newton steps (two: relative error ~1e-15 from the seed's 2.4e-7; no fp64
// division or square-root sequence, which cost ~20 dependent instructions each): the per-pixel loss stays an fp64 quantity
__device__ __forceinline__ double dsqrt_newton(double x) {
  if (!(x > 1e-30 && x < 1e30)) return sqrt(x);
  double r = (double)rsqrtf((float)x);
  r = r * (1.5 - 0.5 * x * r * r);
  r = r * (1.5 - 0.5 * x * r * r);
  return x * r;
}
__device__ __forceinline__ double drecip_newton(double d) {       // d > 0
  if (!(d > 1e-30 && d < 1e30)) return 1.0 / d;                   // outside the float32 seed's comfortable range
  double y = (double)__fdividef(1.0f, (float)d);                   // MUFU.RCP seed: no slow-path subroutine
  y = y * (2.0 - d * y);
  y = y * (2.0 - d * y);
  return y;
}
// per-pixel loss l and detector weight w = dl/dI (readings R11, R12, R12b), fp64
__device__ __forceinline__ void pixel_loss(int loss, double Im, double Ix, double eps, double c, double& l, double& w) {
  if (loss == PT_LOSS_GAUSSIAN) {
    const double ic2 = drecip_newton(c * c);
    l = 0.5 * (Im - Ix) * (Im - Ix) * ic2;
    w = (Im - Ix) * ic2;
  } else if (loss == PT_LOSS_POISSON) {
    const double ri = drecip_newton(Im + eps);
    l = Im - Ix * (1.0 - log((Ix + eps) * ri));                  // = Im - Ix (ln(Im+eps) - ln(Ix+eps) + 1)
    w = 1.0 - Ix * ri;
  } else {
    const double a = dsqrt_newton(Im + c), ae = dsqrt_newton(Ix + c);
    l = 0.5 * (a - ae) * (a - ae);
    w = 0.5 * (1.0 - ae * drecip_newton(a + eps));
  }
}

// The same in float32, written so that no difference of nearly equal numbers is formed from ROUNDED quantities other than the
// inputs themselves (used by the fused single-slice kernel, whose one CTA per SM cannot hide the latency of fp64 sequences — the
// fp64 pipe of this GPU runs at a small fraction of the fp32 rate; the sum over pixels is still taken in fp64):
//   amplitude: d = sqrt(I+c) - sqrt(Iexp+c) ; l = d^2 / 2 ; w = (d + eps) / (2 (sqrt(I+c) + eps))   [= (1 - ae/(a+eps)) / 2]
//   Poisson:   u = (I - Iexp) / (Iexp + eps) ; l = (I - Iexp) - Iexp log1p(u) ; w = (I - Iexp + eps) / (I + eps)
// float32 square root (x >= 0) and reciprocal (d > 0, normal range) from the MUFU seeds and one Newton step each: within an ulp,
// and without the slow-path subroutines of sqrtf() and "/" (taken for zeros, of which a diffraction pattern has many: the loop over
// a thread's 32 pixels cost 33 k cycles with them, 250 instructions per pixel)
__device__ __forceinline__ float sqrt_newton_f32(float x) {
  const float r = rsqrtf(x), a0 = x * r;
  return x > 0.f ? fmaf(0.5f * r, fmaf(-a0, a0, x), a0) : 0.f;
}
__device__ __forceinline__ float rcp_newton_f32(float d) {
  const float y = __fdividef(1.0f, d);
  return y * fmaf(-d, y, 2.0f);
}
__device__ __forceinline__ void pixel_loss_f32(int loss, float Im, float Ix, float eps, float c, float& l, float& w) {
  if (loss == PT_LOSS_GAUSSIAN) {
    const float ic2 = rcp_newton_f32(c * c), d = Im - Ix;
    l = 0.5f * d * d * ic2; w = d * ic2;
  } else if (loss == PT_LOSS_POISSON) {
    const float d = Im - Ix;
    l = d - Ix * log1pf(d * rcp_newton_f32(Ix + eps));
    w = (d + eps) * rcp_newton_f32(Im + eps);
  } else {
    const float a = sqrt_newton_f32(Im + c), d = a - sqrt_newton_f32(Ix + c);
    l = 0.5f * d * d;
    w = 0.5f * (d + eps) * rcp_newton_f32(a + eps);
  }
}

// ------------------------------------------------------------------------------------------------
// H7 + H8: I = sum_k |psi~_k|^2 ; per-pixel loss in fp64 ; w = dl/dI.  One CTA per (position of the chunk, rank).
// ------------------------------------------------------------------------------------------------
template <class G>
__global__ void __launch_bounds__(G::T, 3) k_loss(KP P, float* model_intensity, int want_w) {   // 3 CTAs per SM at T = 512 (40 registers): 1.28 -> 1.13 ms per step at config 3
  typedef Lay<G> L; typedef FL<G> F;
  constexpr int NF = F::NF, NNS = F::NNS, CL = G::CL;
  __shared__ double red[(G::T / 32) * 1];
  const int t = threadIdx.x, jl = blockIdx.x / CL, rk = blockIdx.x - jl * CL, jb = P.j0 + jl;
  const int row = P.w.rows[jb];
  float I[32];
#pragma unroll
  for (int r = 0; r < 32; ++r) I[r] = 0.f;
  for (int k = 0; k < P.M; ++k) {
    const cf* ps = P.w.psit + (((size_t)jl * P.M + k) * CL + rk) * NNS;
#pragma unroll
    for (int r = 0; r < 32; ++r) { cf z = ps[L::native(t, r)]; I[r] = fmaf(z.x, z.x, fmaf(z.y, z.y, I[r])); }
  }
  double acc[1] = {0.0};
  const float* Ie = P.intensity ? P.intensity + (size_t)row * F::NNF : nullptr;
  const double eps = (double)P.eps, c = (double)P.loss_c;
#pragma unroll 4
  for (int r = 0; r < 32; ++r) {
    const int qy = F::fq_y(rk, t, r), qx = F::fq_x(rk, t, r);
    if (model_intensity) model_intensity[(size_t)jb * F::NNF + qy * NF + qx] = I[r];
    if (Ie) {
      const double Im = (double)I[r], Ix = (double)Ie[qy * NF + qx];
      double l, w;
      pixel_loss(P.loss, Im, Ix, eps, c, l, w);
      acc[0] += l;
      if (want_w) P.w.wdet[((size_t)jl * CL + rk) * NNS + L::native(t, r)] = (float)w;
    }
  }
  block_sum<G::T, 1>(acc, red);
  if (t == 0) {
    P.w.loss_pp[(size_t)jb * CL + rk] = acc[0];
    if (!(acc[0] == acc[0]) || fabs(acc[0]) > 1e300) atomicOr(P.w.status, kStatusNonfinite);
  }
}

// ------------------------------------------------------------------------------------------------
// H9, H10, H12, H13 backward: one CTA (CL = 4: one cluster) per (j,k) pair of the chunk: writes the patch-gradient partials
// gT_i, the probe partial conj(R) G~ and the position-gradient terms.  MODE 0: gradients; MODE 2: ePIE directions (R23).
// IL: also stage |Psi_{i,k}|^2 (illumination map O12; denominators of the step-size sweep).
// ------------------------------------------------------------------------------------------------
template <class G, int MODE, bool IL, bool H16>   // H16: the stash holds binary16 pairs (PT_STASH_FP16)
__global__ void __launch_bounds__(G::T, min_blocks<G>()) k_backward(KP P, int want_pos) {
  typedef Lay<G> L; typedef FL<G> F;
  constexpr int NF = F::NF, NNS = F::NNS, T = G::T, E = G::PF16, CL = G::CL;   // stash pairs [0,E) early, [E,16) late; T pairs [0,E) late
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int t = threadIdx.x;
  const unsigned rk = Fft<G>::rank();
  ChainSmem<G> cs(smem_raw, t);
  cf* sm = cs.sm; cf* tw = cs.tw; double* red = cs.red;
  cs.fill_tables(t);
  Fft<G>::begin_fourier();
  const int pair = blockIdx.x / CL, jl = pair / P.M, k = pair - jl * P.M, jb = P.j0 + jl;
  const int spair = pair;
  const int unit = (jb * P.M + k) * CL + (int)rk;                 // index of this CTA's fp64 partials
  const int r0y = P.w.r0[2 * jb], r0x = P.w.r0[2 * jb + 1];
  // patch source: the object window itself, or (bilinear mode) this position's resampled patches [S][NF][NF]
  const int S = P.S, onx = P.bilinear ? NF : P.onx;
  const size_t slice = P.bilinear ? (size_t)F::NNF : (size_t)P.ony * P.onx;
  auto fld = [&](int pr, int i) { return (((size_t)pr * S + i) * CL + rk) * NNS; };   // field (index pr, slice i), this rank's block
  const size_t pix0 = (size_t)F::pix_y(rk, t, 0) * onx + F::pix_x(rk, t, 0);
  const float4* ob2 = (P.bilinear ? P.w.Tb + (size_t)jl * S * F::NNF : P.w.O2 + ((size_t)r0y * P.onx + r0x)) + pix0;   // first pixel with its partner
  // stash pairs [0, E) of slice i one FFT pair ahead; hy table of the propagation that ends iteration i
  auto early = [&](int i) {
    const float4* st = (const float4*)(P.w.stash + fld(pair, i) / (H16 ? 2 : 1)) + t;
    // (the early part itself, pairs [0, E) or the whole binary16 field, arrives by one bulk copy: early_bulk, as in k_backward_pair)
    if (!H16 && t < (16 - E) * T / 8) l2_prefetch_line((const char*)(st - t + E * T) + t * 128);   // the late part of the same field: DRAM -> L2 now, one line per thread
    if (i > 0 && t < NF) {
      cp_async8(cs.hyS + ((i - 1) & 1) * NF + t, P.w.hy + (size_t)(i - 1) * NF + t);
      if (G::HXS) cp_async8(cs.hxS + ((i - 1) & 1) * NF + t, P.w.hx + (size_t)(i - 1) * NF + t);
    }
    cp_async_commit();
  };
  uint64_t* bar = (uint64_t*)((unsigned char*)red + 512);
  auto early_bulk = [&](int i) { bulk_load(cs.pf - t, P.w.stash + fld(pair, i) / (H16 ? 2 : 1), (H16 ? 8 : E) * T * 16, bar); };
  if (t == 0) mbar_init(bar, 1);
  early(S - 1);
  __syncthreads();
  if (t == 0) early_bulk(S - 1);
  cf v[32];
  {   // H9: g~ = w .* psi~ ; gPhi_{S-1} = N Finv(g~) = F^H(g~) / N
    const float4* ps = (const float4*)(P.w.psit + ((size_t)pair * CL + rk) * NNS);
    const float2* wd = (const float2*)(P.w.wdet + ((size_t)jl * CL + rk) * NNS);
    const float sc = (MODE == 2 ? -2.0f : 1.0f) / (float)NF;     // ePIE: chi~ = (ae/(eps+a) - 1) psi~ = -2 w psi~
#pragma unroll
    for (int p = 0; p < 16; ++p) {
      const float4 q = ps[p * T + t]; const float2 w = wd[p * T + t];
      v[2 * p] = make_float2(q.x * (w.x * sc), q.y * (w.x * sc));
      v[2 * p + 1] = make_float2(q.z * (w.y * sc), q.w * (w.y * sc));
    }
  }
  for (int i = S - 1; i >= 0; --i) {
    Fft<G>::inv_head(v, sm, cs.tw2, t, rk);
    const float4* o2 = ob2 + (size_t)i * slice;
    float4 Tr[H16 ? 1 : 16 - E];                                  // patch pairs [E, 16): no slot left in shared memory
    if (H16) {   // late: all of T_i into the warp's idle X1 region (the stash is in the early slots)
#pragma unroll
      for (int p = 0; p < 16; ++p) cp_async16(cs.xs + p * 32, o2 + F::patch_off(2 * p, onx));
      cp_async_commit();
      L::phase1_inv(v, tw, t);                                   // gPhi_{i,k}  (R-layout)
    } else {
      // late: the rest of the stash and T pairs [0, E) into the warp's idle X1 region, T registers [2E, 32) (no slot left in shared
      // memory) by plain loads: 22 instructions per thread, a few between the steps of phase 1 instead of one burst before it
      const float4* st = (const float4*)(P.w.stash + fld(pair, i)) + t;
      constexpr int NQ = (16 - E) + E + (16 - E), NH = G::N1X + G::N1Y;
      auto item = [&](int q) {
        if (q < 16 - E) cp_async16(cs.xs + q * 32, st + (E + q) * T);
        else if (q < 16) { const int p = q - (16 - E); cp_async16(cs.xs + (16 - E + p) * 32, o2 + F::patch_off(2 * p, onx)); }
        else { const int p = E + (q - 16); Tr[p - E] = ld_nc16(o2 + F::patch_off(2 * p, onx)); }
      };
      constexpr int NHU = NH * 2 / 3;                              // within the first two thirds of the steps (see k_backward_pair)
      L::phase1_inv_h(v, tw, t, [&](int step) {                  // gPhi_{i,k}  (R-layout)
#pragma unroll
        for (int q = 0; q < NQ; ++q) if (q * NHU / NQ == step) item(q);
      });
      cp_async_commit();
    }
    cp_async_wait_all();
    mbar_wait(bar, (unsigned)((S - 1 - i) & 1));                 // the early part of this slice's stash field has landed
    // ePIE (MODE 2): dO = conj(Psi) / max|Psi|^2 chi ; chi' = conj(T) / max|T|^2 chi
    float s1 = 1.0f, s2 = 1.0f;
    if (MODE == 2) {
      float pm = 0.f;
      for (int c = 0; c < CL; ++c) pm = fmaxf(pm, P.w.psimax[((size_t)pair * S + i) * CL + c]);
      const float tm = P.w.tmax[(size_t)jl * S + i];
      s1 = pm > 0.f ? 1.0f / pm : 0.f; s2 = tm > 0.f ? 1.0f / tm : 0.f;   // a dead mode / an opaque window contributes nothing (R23b)
    }
    float4* gt = (float4*)(P.w.gTpart + fld(spair, i));
    float2* il = IL ? (float2*)(P.w.ilpart + fld(spair, i)) : nullptr;
    float4 hw = make_float4(0.f, 0.f, 0.f, 0.f);                  // H16: the 16-byte word that holds pairs p, p + 1 (p even)
#pragma unroll
    for (int p = 0; p < 16; ++p) {
      float4 ps;
      cf T0, T1;
      if (H16) {
        if (!(p & 1)) hw = cs.pf[(p >> 1) * T];
        const cf a = unpack_h2(__float_as_uint((p & 1) ? hw.z : hw.x)), b = unpack_h2(__float_as_uint((p & 1) ? hw.w : hw.y));
        ps = make_float4(a.x, a.y, b.x, b.y);
        const float4 tt = cs.xs[p * 32];
        T0 = make_float2(tt.x, tt.y); T1 = make_float2(tt.z, tt.w);
      } else {
        ps = p < E ? cs.pf[p * T] : cs.xs[(p - E) * 32];
        const float4 tt = p < E ? cs.xs[(16 - E + p) * 32] : Tr[p - E];
        T0 = make_float2(tt.x, tt.y); T1 = make_float2(tt.z, tt.w);
      }
      cf g0 = cmulc(v[2 * p], make_float2(ps.x, ps.y)), g1 = cmulc(v[2 * p + 1], make_float2(ps.z, ps.w));
      if (MODE == 2) { g0 = cscale(g0, s1); g1 = cscale(g1, s1); T0 = cscale(T0, s2); T1 = cscale(T1, s2); }
      if (IL) __stcs(il + p * T + t, make_float2(fmaf(ps.x, ps.x, ps.y * ps.y), fmaf(ps.z, ps.z, ps.w * ps.w)));
      __stcs(gt + p * T + t, make_float4(g0.x, g0.y, g1.x, g1.y));    // H10: gT_i contribution conj(Psi) .* gPhi
      v[2 * p] = cmulc(v[2 * p], T0);                          //      gPsi = conj(T) .* gPhi
      v[2 * p + 1] = cmulc(v[2 * p + 1], T1);
    }
    if (i > 0) early(i - 1);
    Fft<G>::fwd(v, sm, tw, cs.tw2, t, rk);                       // F(gPsi_i)  (Fourier layout)
    if (t == 0 && i > 0) early_bulk(i - 1);                      // behind the forward transform's last CTA barrier: every thread has read its slots
    if (i > 0) apply_prop_t<G, true>(v, G::HXS ? cs.hxS + ((i - 1) & 1) * NF : P.w.hx + (size_t)(i - 1) * NF, cs.hyS + ((i - 1) & 1) * NF, P.bandlim2, t, rk);
  }
  const cf* rx = P.w.ramps + (size_t)jb * 2 * NF;
  const cf* ry = rx + NF;
  const cf* pt = P.w.Pt + ((size_t)k * CL + rk) * NNS;
  // v = G~ = F(gPsi_0).  H12: probe partial conj(R) .* G~ ;  H13: (4 pi / N^2) sum_q f_a Im(conj(G~) R P~)
  cf* gp = P.w.Gpart + ((size_t)spair * CL + rk) * NNS;
  cf wxv[F::NXV];
  load_xv<G>(wxv, rx, t, 1.0f);
  float sy = 0.f, sx = 0.f;
#pragma unroll
  for (int r = 0; r < 32; ++r) {
    const int qy = F::fq_y(rk, t, r);
    const cf R = cmul(wxv[F::fq_xsel(r)], ry[qy]);
    gp[L::native(t, r)] = cmulc(v[r], R);
    if (want_pos) {
      const cf z = cmulc(cmul(R, pt[L::native(t, r)]), v[r]);  // conj(G~) R P~
      const float fy = (float)signed_freq(qy, NF) / (float)NF, fx = (float)signed_freq(F::fq_x(rk, t, r), NF) / (float)NF;
      sy = fmaf(fy, z.y, sy); sx = fmaf(fx, z.y, sx);
    }
  }
  if (want_pos) {
    double acc[2] = {(double)sy, (double)sx};
    block_sum<G::T, 2>(acc, red);
    if (t == 0) {
      const double f = 4.0 * CUDART_PI / ((double)NF * (double)NF);
      P.w.posg_part[(size_t)unit * 2 + 0] = f * acc[0];
      P.w.posg_part[(size_t)unit * 2 + 1] = f * acc[1];
    }
  }
  Fft<G>::end_fourier();
}

// ------------------------------------------------------------------------------------------------
// H14, LSQML-style step-size terms from what the gradient pass has staged.  With
// chi_{i,k} = -c gPhi_{i,k} (c = KP::chi_scale) and u = dOhat|patch .* Psi_{i,k}:
//   numO_i = sum_{k,r} Re(chi conj(u)) = -c Re sum_r conj(dOhat[r0 + r]) sum_k gT_{i,k}[r]        (gT = conj(Psi) gPhi, staged)
//   denO_i = sum_{k,r} |u|^2          = sum_r |dOhat[r0 + r]|^2 sum_k |Psi_{i,k}[r]|^2            (|Psi|^2 staged)
// i.e. the sums of the paper's formula in another order: no second pass through the FFT chain.  One block per (position of
// the chunk, slice); fp64 sums in fixed order.  Bilinear mode (R1, R30): dOhat is sampled with the four taps, and the position
// terms come through the patch: numX_a = -c Re sum_i sum_r conj(dT_i/df_a) gT_i, denX_a = sum_i sum_r |dT_i/df_a|^2 sum_k |Psi|^2.
// ------------------------------------------------------------------------------------------------
template <class G, bool BILIN>
__global__ void __launch_bounds__(256) k_step_object(KP P) {
  typedef Lay<G> L; typedef FL<G> F;
  constexpr int NNS = F::NNS, T = G::T, CL = G::CL, NV = BILIN ? 6 : 2;
  __shared__ double red[(256 / 32) * NV];
  const int jl = blockIdx.x / P.S, i = blockIdx.x - jl * P.S, jb = P.j0 + jl, sj = jl;
  const int r0y = P.w.r0[2 * jb], r0x = P.w.r0[2 * jb + 1];
  const size_t onx = P.onx;
  const cf* dO = P.w.dOhat + ((size_t)i * P.ony + r0y) * onx + r0x;
  const cf* ob = P.object + ((size_t)i * P.ony + r0y) * onx + r0x;
  float w00 = 1.f, w01 = 0.f, w10 = 0.f, w11 = 0.f, fy = 0.f, fx = 0.f;
  if (BILIN) {
    fy = P.w.delta[2 * jb]; fx = P.w.delta[2 * jb + 1];
    w00 = (1.f - fy) * (1.f - fx); w01 = (1.f - fy) * fx; w10 = fy * (1.f - fx); w11 = fy * fx;
  }
  double acc[NV];
#pragma unroll
  for (int c = 0; c < NV; ++c) acc[c] = 0.0;
  for (int e = threadIdx.x; e < CL * NNS; e += 256) {              // e: element of the field in storage order [rank][native]
    const int rank = e / NNS, n = e - rank * NNS, m = n >> 1, t = m % T, r = ((m / T) << 1) | (n & 1);
    const int y = F::pix_y(rank, t, r), x = F::pix_x(rank, t, r);
    double gr = 0.0, gi = 0.0, il = 0.0;
    const size_t gb = ((size_t)sj * P.Mg * P.S + i) * (CL * NNS) + e;
    for (int k = 0; k < P.Mg; ++k) { const cf g = P.w.gTpart[gb + (size_t)k * P.S * (CL * NNS)]; gr += (double)g.x; gi += (double)g.y; }
    const size_t ib = ((size_t)sj * P.Mi * P.S + i) * (CL * NNS) + e;
    for (int k = 0; k < P.Mi; ++k) il += (double)P.w.ilpart[ib + (size_t)k * P.S * (CL * NNS)];
    const size_t o = (size_t)y * onx + x;
    double dr, di;
    if (BILIN) {
      const cf a = dO[o], b = dO[o + 1], c = dO[o + onx], d = dO[o + onx + 1];
      dr = (double)(w00 * a.x + w01 * b.x + w10 * c.x + w11 * d.x); di = (double)(w00 * a.y + w01 * b.y + w10 * c.y + w11 * d.y);
      const cf oa = ob[o], obb = ob[o + 1], oc = ob[o + onx], od = ob[o + onx + 1];
      const double tyr = (1.0 - fx) * ((double)oc.x - oa.x) + fx * ((double)od.x - obb.x), tyi = (1.0 - fx) * ((double)oc.y - oa.y) + fx * ((double)od.y - obb.y);
      const double txr = (1.0 - fy) * ((double)obb.x - oa.x) + fy * ((double)od.x - oc.x), txi = (1.0 - fy) * ((double)obb.y - oa.y) + fy * ((double)od.y - oc.y);
      acc[2] -= tyr * gr + tyi * gi; acc[3] += (tyr * tyr + tyi * tyi) * il;
      acc[4] -= txr * gr + txi * gi; acc[5] += (txr * txr + txi * txi) * il;
    } else {
      const cf d = dO[o];
      dr = (double)d.x; di = (double)d.y;
    }
    acc[0] -= dr * gr + di * gi;                                    // -Re(conj(dOhat) gT)
    acc[1] += (dr * dr + di * di) * il;
  }
  block_sum<256, NV>(acc, red);
  if (threadIdx.x == 0) {
    const double c = (double)P.chi_scale;
    double* out = P.w.step_oi + ((size_t)jb * P.S + i) * 6;
    out[0] = c * c * acc[0]; out[1] = c * c * acc[1];               // dOhat carries one factor c, chi the other
#pragma unroll
    for (int q = 2; q < 6; ++q) out[q] = 0.0;
    if (BILIN) { out[2] = c * acc[2]; out[3] = acc[3]; out[4] = c * acc[4]; out[5] = acc[5]; }
  }
}

// Probe and (Fourier-shift mode) position terms of the step-size sweep, one CTA (cluster) per (position of the chunk, mode).
// With G~ = F(conj(T_0) gPhi_0) from the gradient pass (staged as Gpart = conj(R) G~) the numerators are dot products on the
// Fourier side (Parseval):  numP = -c^2/N^2 Re sum_q conj(Q~_k) Gpart,  numX_a = c 2 pi / N^2 sum_q f_a Im(conj(P~_k) Gpart);
// the denominators need the fields in real space: denP = c^2 sum_r |shift_j(dPhat_k) T_0|^2, denX_a = sum_r |dPsi_0/d delta_a T_0|^2
// — three inverse transforms instead of a second pass through the 2S transforms of the chain.
template <class G>
__global__ void __launch_bounds__(G::T, min_blocks<G>()) k_step_probe(KP P) {
  typedef Lay<G> L; typedef FL<G> F;
  constexpr int NF = F::NF, NNS = F::NNS, CL = G::CL;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int t = threadIdx.x;
  const unsigned rk = Fft<G>::rank();
  ChainSmem<G> cs(smem_raw, t);
  cf* sm = cs.sm; cf* tw = cs.tw; double* red = cs.red;
  cs.fill_tables(t);
  const int pair = blockIdx.x / CL, jl = pair / P.M, k = pair - jl * P.M, jb = P.j0 + jl;
  const int spair = pair;
  const int r0y = P.w.r0[2 * jb], r0x = P.w.r0[2 * jb + 1];
  const int onx = P.bilinear ? NF : P.onx;
  const size_t pix0 = (size_t)F::pix_y(rk, t, 0) * onx + F::pix_x(rk, t, 0);     // this thread's first pixel
  const cf* ob = patch_ptr(P, 0, r0y, r0x) + pix0;                               // T_0: the object window, or (bilinear mode) the first
  const float4* ob2 = P.bilinear ? P.w.Tb + (size_t)jl * P.S * F::NNF + pix0 : nullptr;   // halves of this position's sampled pairs
  const cf* rx = P.w.ramps + (size_t)jb * 2 * NF;
  const cf* ry = rx + NF;
  const cf* pt = P.w.Pt + ((size_t)k * CL + rk) * NNS;
  const cf* qt = P.w.Qt + ((size_t)k * CL + rk) * NNS;
  const cf* gp = P.w.Gpart + ((size_t)spair * CL + rk) * NNS;
  const double c = (double)P.chi_scale, inn = 1.0 / ((double)NF * (double)NF);
  double* sp = P.w.step_pp + ((size_t)(jb * P.M + k) * CL + rk) * 6;
  __syncthreads();
  {   // numerators
    float np = 0.f, ny = 0.f, nx = 0.f;
#pragma unroll
    for (int r = 0; r < 32; ++r) {
      const cf g = gp[L::native(t, r)], q = qt[L::native(t, r)], pp = pt[L::native(t, r)];
      np -= fmaf(q.x, g.x, q.y * g.y);                               // -Re(conj(Q~) Gpart)
      const float im = fmaf(pp.x, g.y, -(pp.y * g.x));              // Im(conj(P~) Gpart)
      ny = fmaf((float)signed_freq(F::fq_y(rk, t, r), NF) / (float)NF, im, ny);
      nx = fmaf((float)signed_freq(F::fq_x(rk, t, r), NF) / (float)NF, im, nx);
    }
    double acc[3] = {(double)np, (double)ny, (double)nx};
    block_sum<G::T, 3>(acc, red);
    if (t == 0) { sp[0] = c * c * inn * acc[0]; sp[2] = c * 2.0 * CUDART_PI * inn * acc[1]; sp[4] = c * 2.0 * CUDART_PI * inn * acc[2]; }
  }
  cf wxv[F::NXV];
  load_xv<G>(wxv, rx, t, 1.0f / (float)F::NNF);
  const int nterm = P.bilinear ? 1 : 3;                             // bilinear mode: the position terms come from k_step_object
  cf v[32];
  for (int term = 0; term < nterm; ++term) {
#pragma unroll
    for (int r = 0; r < 32; ++r) {
      const int qy = F::fq_y(rk, t, r);
      const cf R = cmul(wxv[F::fq_xsel(r)], ry[qy]);
      if (term == 0) v[r] = cmul(R, qt[L::native(t, r)]);                       // shift_j(dPhat_k)
      else {
        const float f = (float)signed_freq(term == 1 ? qy : F::fq_x(rk, t, r), NF) / (float)NF;   // d Psi_0 / d delta_a
        const cf z = cmul(R, pt[L::native(t, r)]);
        const float g = -2.0f * CUDART_PI_F * f;
        v[r] = make_float2(-g * z.y, g * z.x);                                  // (i g) z
      }
    }
    Fft<G>::begin_fourier();
    Fft<G>::inv(v, sm, tw, cs.tw2, t, rk);
    float den = 0.f;
#pragma unroll
    for (int r = 0; r < 32; ++r) {
      cf T0;
      if (P.bilinear) { const float4 q = ob2[F::patch_off(r, onx)]; T0 = make_float2(q.x, q.y); }
      else T0 = ob[F::patch_off(r, onx)];
      const cf u = cmul(v[r], T0);
      den = fmaf(u.x, u.x, fmaf(u.y, u.y, den));
    }
    double acc[1] = {(double)den};
    block_sum<G::T, 1>(acc, red);
    if (t == 0) sp[2 * term + 1] = (term == 0 ? c * c : 1.0) * acc[0];
    __syncthreads();
  }
  if (t == 0 && P.bilinear) { sp[2] = 0.0; sp[3] = 0.0; sp[4] = 0.0; sp[5] = 0.0; }
}

// ------------------------------------------------------------------------------------------------
// Tensor memory (TMEM, 256 KB per SM, otherwise unused by this library) as a per-thread parking space: a warp may touch
// the 32 lanes of its own quarter (warp % 4) and any column; each warp gets 128 columns (64 for a parked field, 64 for the
// first mode's patch gradient).  Measured on B200 (148 CTAs x 512 threads): swapping 64 registers per thread with TMEM costs
// 576 cycles per CTA, a 64-register load 371.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void tmem_st4(uint32_t a, cf x, cf y) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(__float_as_uint(x.x)), "r"(__float_as_uint(x.y)),
               "r"(__float_as_uint(y.x)), "r"(__float_as_uint(y.y)) : "memory");
}
__device__ __forceinline__ void tmem_ld4(uint32_t a, cf& x, cf& y) {
  uint32_t r0, r1, r2, r3;
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(a) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
  x = make_float2(__uint_as_float(r0), __uint_as_float(r1)); y = make_float2(__uint_as_float(r2), __uint_as_float(r3));
}
__device__ __forceinline__ void tmem_st16(uint32_t a, const cf* v) {   // 8 complex = 16 columns
  asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(a),
               "r"(__float_as_uint(v[0].x)), "r"(__float_as_uint(v[0].y)), "r"(__float_as_uint(v[1].x)), "r"(__float_as_uint(v[1].y)),
               "r"(__float_as_uint(v[2].x)), "r"(__float_as_uint(v[2].y)), "r"(__float_as_uint(v[3].x)), "r"(__float_as_uint(v[3].y)),
               "r"(__float_as_uint(v[4].x)), "r"(__float_as_uint(v[4].y)), "r"(__float_as_uint(v[5].x)), "r"(__float_as_uint(v[5].y)),
               "r"(__float_as_uint(v[6].x)), "r"(__float_as_uint(v[6].y)), "r"(__float_as_uint(v[7].x)), "r"(__float_as_uint(v[7].y)) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t a, cf* v) {
  uint32_t r[16];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
                 "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]) : "r"(a) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 8; ++i) v[i] = make_float2(__uint_as_float(r[2 * i]), __uint_as_float(r[2 * i + 1]));
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_st8(uint32_t a, const cf* v) {   // 4 complex = 8 columns
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(a),
               "r"(__float_as_uint(v[0].x)), "r"(__float_as_uint(v[0].y)), "r"(__float_as_uint(v[1].x)), "r"(__float_as_uint(v[1].y)),
               "r"(__float_as_uint(v[2].x)), "r"(__float_as_uint(v[2].y)), "r"(__float_as_uint(v[3].x)), "r"(__float_as_uint(v[3].y)) : "memory");
}
__device__ __forceinline__ void tmem_ld8(uint32_t a, cf* v) {
  uint32_t r[8];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "r"(a) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 4; ++i) v[i] = make_float2(__uint_as_float(r[2 * i]), __uint_as_float(r[2 * i + 1]));
}
// v <-> parked field (columns [0, 64) of the warp's block), four complex at a time.  Sixteen-column accesses want sixteen
// CONSECUTIVE registers on both sides: with them the register allocator spilled one quarter of the incoming field in every half step
// (16 LDL + 8 STL.64, 4.6 % of the kernel's stall samples; ncu source page); eight-column accesses leave 8 bytes of spill and the
// backward kernel runs 52.4 -> 50.0 ms per step at config 3.
__device__ __forceinline__ void tmem_swap_field(uint32_t tb, cf (&v)[32]) {
#pragma unroll
  for (int c = 0; c < 8; ++c) {
    cf tmp[4];
    tmem_ld8(tb + c * 8, tmp);
    tmem_st8(tb + c * 8, &v[4 * c]);
#pragma unroll
    for (int i = 0; i < 4; ++i) v[4 * c + i] = tmp[i];
  }
  tmem_wait_st();
}

// ------------------------------------------------------------------------------------------------
// H9, H10, H12, H13 backward for TWO modes per CTA (or cluster of four at N = 256); M even: the two adjoint chains advance slice by slice in turn,
// the field of the mode that is not being worked on parked in TMEM, so that the patch gradients of the pair are summed on
// chip (first mode's gT_i kept in TMEM until the second mode reaches slice i) and only the sum goes to the staging buffer:
// half the staging writes here and half the reads in k_gather_object.  Same arithmetic per mode as k_backward (MODE 0 / 2);
// the sum over the pair is taken in float32 in fixed order (first + second), the gather then sums the pairs in fp64.
// Staging layout: [Jc][M/2][S][N^2].
// ------------------------------------------------------------------------------------------------
template <class G, int MODE, bool IL, bool H16>   // IL: also stage |Psi_{i,k}|^2 (O12); H16: the stash holds binary16 pairs (PT_STASH_FP16)
__global__ void __launch_bounds__(G::T, min_blocks<G>()) k_backward_pair(KP P, int want_pos) {
  typedef Lay<G> L; typedef FL<G> F;
  constexpr int NF = F::NF, NNS = F::NNS, T = G::T, E = G::PF16, CL = G::CL, TCOLS = T;       // T/32 warps, 4 per lane quarter, 128 columns each
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int t = threadIdx.x, wp = t >> 5;
  const unsigned rk = Fft<G>::rank();
  ChainSmem<G> cs(smem_raw, t);
  cf* sm = cs.sm; cf* tw = cs.tw; double* red = cs.red;
  uint32_t* tmem_slot = (uint32_t*)((unsigned char*)red + 1000);                  // beyond what block_sum uses of the 1 KB scratch
  cs.fill_tables(t);
  Fft<G>::begin_fourier();
  if (wp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(tmem_slot)), "n"(TCOLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  const int MP = P.M >> 1, pp = blockIdx.x / CL, jl = pp / MP, kp = pp - jl * MP, jb = P.j0 + jl;
  const int pair0 = jl * P.M + 2 * kp;                                            // (position, mode) index of the pair's first mode
  const int r0y = P.w.r0[2 * jb], r0x = P.w.r0[2 * jb + 1];
  const int S = P.S, onx = P.bilinear ? NF : P.onx;
  const size_t slice = P.bilinear ? (size_t)F::NNF : (size_t)P.ony * P.onx;
  auto fld = [&](int pr, int i) { return (((size_t)pr * S + i) * CL + rk) * NNS; };   // field (index pr, slice i), this rank's block
  const size_t pix0 = (size_t)F::pix_y(rk, t, 0) * onx + F::pix_x(rk, t, 0);
  const float4* ob2 = (P.bilinear ? P.w.Tb + (size_t)jl * S * F::NNF : P.w.O2 + ((size_t)r0y * P.onx + r0x)) + pix0;   // first pixel with its partner
  // half step s = 0 .. 2S-1: mode h = s & 1 of the pair at slice i = S-1 - (s >> 1)
  auto early = [&](int s) {
    const int h = s & 1, i = S - 1 - (s >> 1);
    const float4* st = (const float4*)(P.w.stash + fld(pair0 + h, i) / (H16 ? 2 : 1)) + t;
    // (the early part itself, pairs [0, E) or the whole binary16 field, arrives by ONE bulk copy: early_bulk below)
    if (!H16 && t < (16 - E) * T / 8) l2_prefetch_line((const char*)(st - t + E * T) + t * 128);   // the late part of the same field: DRAM -> L2 now, one line per thread
    if (h == 0 && i > 0 && t < NF) {                              // serves both modes at slice i
      cp_async8(cs.hyS + ((i - 1) & 1) * NF + t, P.w.hy + (size_t)(i - 1) * NF + t);
      if (G::HXS) cp_async8(cs.hxS + ((i - 1) & 1) * NF + t, P.w.hx + (size_t)(i - 1) * NF + t);
    }
    cp_async_commit();
  };
  // The early slots of all threads are one contiguous block [pair][thread] in shared memory and in the stash, so ONE bulk copy
  // (cp.async.bulk, completion on an mbarrier) issued by thread 0 replaces ten 16-byte cp.async per thread (backward 53.9 -> 53.1 ms
  // per step).  It overwrites every thread's slots: issued behind a CTA barrier that follows their last readers.
  uint64_t* bar = (uint64_t*)((unsigned char*)red + 512);
  auto early_bulk = [&](int s) {
    const int h = s & 1, i = S - 1 - (s >> 1);
    bulk_load(cs.pf - t, P.w.stash + fld(pair0 + h, i) / (H16 ? 2 : 1), (H16 ? 8 : E) * T * 16, bar);
  };
  if (t == 0) mbar_init(bar, 1);
  early(0);
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  if (t == 0) early_bulk(0);
  const uint32_t tb = *tmem_slot + ((uint32_t)((wp & 3) * 32) << 16) + (uint32_t)((wp >> 2) * 128);
  cf v[32];
  auto init = [&](int pr) {   // H9: g~ = w .* psi~ ; gPhi_{S-1} = F^H(g~) / N
    const float4* ps = (const float4*)(P.w.psit + ((size_t)pr * CL + rk) * NNS);
    const float2* wd = (const float2*)(P.w.wdet + ((size_t)jl * CL + rk) * NNS);
    const float sc = (MODE == 2 ? -2.0f : 1.0f) / (float)NF;
#pragma unroll
    for (int p = 0; p < 16; ++p) {
      const float4 q = ps[p * T + t]; const float2 w = wd[p * T + t];
      v[2 * p] = make_float2(q.x * (w.x * sc), q.y * (w.x * sc));
      v[2 * p + 1] = make_float2(q.z * (w.y * sc), q.w * (w.y * sc));
    }
  };
  init(pair0 + 1);
#pragma unroll
  for (int c = 0; c < 4; ++c) tmem_st16(tb + c * 16, &v[8 * c]);                  // park the second mode
  tmem_wait_st();
  init(pair0);
#pragma unroll 1
  for (int s = 0; s < 2 * S; ++s) {
    const int h = s & 1, i = S - 1 - (s >> 1), pr = pair0 + h;
    Fft<G>::inv_head(v, sm, cs.tw2, t, rk);
    const float4* o2 = ob2 + (size_t)i * slice;
    float4 Tr[H16 ? 1 : 16 - E];                                  // patch pairs [E, 16): no slot left in shared memory
    if (H16) {
#pragma unroll
      for (int p = 0; p < 16; ++p) cp_async16(cs.xs + p * 32, o2 + F::patch_off(2 * p, onx));
      cp_async_commit();
      L::phase1_inv(v, tw, t);
    } else {
      // the late copies and direct loads (22 instructions per thread), a few between the steps of phase 1 instead of one burst before it
      const float4* st = (const float4*)(P.w.stash + fld(pr, i)) + t;
      constexpr int NQ = (16 - E) + E + (16 - E), NH = G::N1X + G::N1Y;
      auto item = [&](int q) {
        if (q < 16 - E) cp_async16(cs.xs + q * 32, st + (E + q) * T);
        else if (q < 16) { const int p = q - (16 - E); cp_async16(cs.xs + (16 - E + p) * 32, o2 + F::patch_off(2 * p, onx)); }
        else { const int p = E + (q - 16); Tr[p - E] = ld_nc16(o2 + F::patch_off(2 * p, onx)); }
      };
      // over the first two thirds of the steps only: spread over all of them, the last copies were issued ~20 instructions before the
      // wait below in some variants (ncu, illumination-staging kernel: 2.3 % of the samples on that wait); 49.8 -> 49.1 ms per step
      constexpr int NHU = NH * 2 / 3;
      L::phase1_inv_h(v, tw, t, [&](int step) {                  // gPhi_{i,k}  (R-layout); backward 56.4 -> 55.5 ms per step
#pragma unroll
        for (int q = 0; q < NQ; ++q) if (q * NHU / NQ == step) item(q);
      });
      cp_async_commit();
    }
    cp_async_wait_all();
    mbar_wait(bar, (unsigned)(s & 1));                           // the early part of this half step's stash field has landed
    float s1 = 1.0f, s2 = 1.0f;
    if (MODE == 2) {
      float pm = 0.f;
      for (int c = 0; c < CL; ++c) pm = fmaxf(pm, P.w.psimax[((size_t)pr * S + i) * CL + c]);
      const float tm = P.w.tmax[(size_t)jl * S + i];
      s1 = pm > 0.f ? 1.0f / pm : 0.f; s2 = tm > 0.f ? 1.0f / tm : 0.f;
    }
    float4* gt = (float4*)(P.w.gTpart + fld(pp, i));
    float2* il = IL ? (float2*)(P.w.ilpart + fld(pp, i)) : nullptr;   // O12 staging: |Psi|^2 summed over the pair (first mode stores, second adds)
    float4 hw = make_float4(0.f, 0.f, 0.f, 0.f);                  // H16: the 16-byte word that holds pairs p, p + 1 (p even)
#pragma unroll
    for (int p = 0; p < 16; ++p) {
      float4 ps;
      cf T0, T1;
      if (H16) {
        if (!(p & 1)) hw = cs.pf[(p >> 1) * T];
        const cf a = unpack_h2(__float_as_uint((p & 1) ? hw.z : hw.x)), b = unpack_h2(__float_as_uint((p & 1) ? hw.w : hw.y));
        ps = make_float4(a.x, a.y, b.x, b.y);
        const float4 tt = cs.xs[p * 32];
        T0 = make_float2(tt.x, tt.y); T1 = make_float2(tt.z, tt.w);
      } else {
        ps = p < E ? cs.pf[p * T] : cs.xs[(p - E) * 32];
        const float4 tt = p < E ? cs.xs[(16 - E + p) * 32] : Tr[p - E];
        T0 = make_float2(tt.x, tt.y); T1 = make_float2(tt.z, tt.w);
      }
      cf g0 = cmulc(v[2 * p], make_float2(ps.x, ps.y)), g1 = cmulc(v[2 * p + 1], make_float2(ps.z, ps.w));
      if (MODE == 2) { g0 = cscale(g0, s1); g1 = cscale(g1, s1); T0 = cscale(T0, s2); T1 = cscale(T1, s2); }
      if (IL) {
        const float i0 = fmaf(ps.x, ps.x, ps.y * ps.y), i1 = fmaf(ps.z, ps.z, ps.w * ps.w);
        if (h == 0) il[p * T + t] = make_float2(i0, i1);         // stays in L2 until the second mode's half step adds to it: the same thread,
        else asm volatile("red.global.add.v2.f32 [%0], {%1,%2};" ::"l"(il + p * T + t), "f"(i0), "f"(i1) : "memory");   // program order, one adder: deterministic
      }
      if (h == 0) tmem_st4(tb + 64 + 4 * p, g0, g1);             // first mode: keep gT_i on chip
      else {                                                     // second mode: the pair's sum goes to the staging buffer
        cf a0, a1;
        tmem_ld4(tb + 64 + 4 * p, a0, a1);
        __stcs(gt + p * T + t, make_float4(a0.x + g0.x, a0.y + g0.y, a1.x + g1.x, a1.y + g1.y));
      }
      v[2 * p] = cmulc(v[2 * p], T0);                            // gPsi = conj(T) .* gPhi
      v[2 * p + 1] = cmulc(v[2 * p + 1], T1);
      if ((p & 3) == 3) L::phase1_fwd_row(v, p >> 2);            // row transform of the eight registers that are final (as in k_forward)
    }
    if (h == 0) tmem_wait_st();
    if (s + 1 < 2 * S) early(s + 1);
    Fft<G>::fwd_after_rows(v, sm, tw, cs.tw2, t, rk);             // F(gPsi_i)
    if (i > 0) apply_prop_t<G, true>(v, G::HXS ? cs.hxS + ((i - 1) & 1) * NF : P.w.hx + (size_t)(i - 1) * NF, cs.hyS + ((i - 1) & 1) * NF, P.bandlim2, t, rk);
    if (t == 0 && s + 1 < 2 * S) early_bulk(s + 1);               // behind the forward transform's last CTA barrier: every thread has read its slots
    tmem_swap_field(tb, v);                                      // the other mode's turn
  }
  // v = G~ of the first mode, the second mode's is parked.  H12 / H13 per mode as in k_backward.
  const cf* rx = P.w.ramps + (size_t)jb * 2 * NF;
  const cf* ry = rx + NF;
#pragma unroll 1
  for (int h = 0; h < 2; ++h) {
    if (h == 1) {
#pragma unroll
      for (int c = 0; c < 4; ++c) tmem_ld16(tb + c * 16, &v[8 * c]);
    }
    const int pr = pair0 + h, k = 2 * kp + h;
    const cf* pt = P.w.Pt + ((size_t)k * CL + rk) * NNS;
    cf* gp = P.w.Gpart + ((size_t)pr * CL + rk) * NNS;
    cf wxv[F::NXV];
    load_xv<G>(wxv, rx, t, 1.0f);
    float sy = 0.f, sx = 0.f;
#pragma unroll
    for (int r = 0; r < 32; ++r) {
      const int qy = F::fq_y(rk, t, r);
      const cf R = cmul(wxv[F::fq_xsel(r)], ry[qy]);
      gp[L::native(t, r)] = cmulc(v[r], R);
      if (want_pos) {
        const cf z = cmulc(cmul(R, pt[L::native(t, r)]), v[r]);
        const float fy = (float)signed_freq(qy, NF) / (float)NF, fx = (float)signed_freq(F::fq_x(rk, t, r), NF) / (float)NF;
        sy = fmaf(fy, z.y, sy); sx = fmaf(fx, z.y, sx);
      }
    }
    if (want_pos) {
      double acc[2] = {(double)sy, (double)sx};
      block_sum<G::T, 2>(acc, red);
      if (t == 0) {
        const double f = 4.0 * CUDART_PI / ((double)NF * (double)NF);
        const size_t unit = ((size_t)jb * P.M + k) * CL + rk;       // index of this CTA's fp64 partials
        P.w.posg_part[unit * 2 + 0] = f * acc[0];
        P.w.posg_part[unit * 2 + 1] = f * acc[1];
      }
    }
  }
  Fft<G>::end_fourier();
  __syncthreads();
  if (wp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(*tmem_slot), "n"(TCOLS));
}

// ------------------------------------------------------------------------------------------------
// Single-slice path (S = 1: BASELINE.json configs 1 and 2; "strong phase object approximation"): forward model, loss
// and adjoint of ONE position in one persistent CTA, all modes in turn — no kernel boundary between H2..H13, no per-mode staging:
//   pass 1, mode k:  Psi_k = Finv(R P~_k)/N^2 -> scratch ; Phi = Psi_k T ; psi~_k = F(Phi)/N -> scratch ; I += |psi~_k|^2
//   loss:            l(I, Iexp) per pixel in fp64, w = dl/dI                                   (as k_loss)
//   pass 2, mode k:  gPhi = F^H(w psi~_k)/N ; gT += conj(Psi_k) gPhi ; G~ = F(conj(T) gPhi) ; probe partial conj(R) G~ ;
//                    position terms                                                            (as k_backward)
// On chip for the whole position: the patch T and the mode sum of gT in tensor memory (64 + 64 columns per warp), I (then w) in
// the thread-private shared-memory slots, the shift ramp ry in the (otherwise idle) propagator-table buffer.  Psi_k and psi~_k
// pass through the per-position scratch of the workspace (the stash / far-field arrays of the chain path; the CTA reads back what
// it wrote shortly before, from L2).  Only ONE patch-gradient plane per position is staged (fp32 sum over the modes in order),
// so the gather reads 1/M of what the per-mode kernels stage, and ONE probe-partial plane per (CTA, mode): the CTA's positions are
// added in float32 in the order it takes them.  CTAs stay resident and take positions jl = blockIdx.x, + gridDim.x, ...
// ------------------------------------------------------------------------------------------------
template <class G>
__global__ void __launch_bounds__(G::T, min_blocks<G>()) k_single(KP P, int want_pos) {
  typedef Lay<G> L; typedef FL<G> F;
  static_assert(G::CL == 1, "single-slice path: one CTA per field");
  constexpr int NF = F::NF, NNS = F::NNS, T = G::T, TCOLS = (T / 128) * 128;     // 128 columns per warp: T and the gT sum
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int t = threadIdx.x, wp = t >> 5;
  ChainSmem<G> cs(smem_raw, t);
  cf* sm = cs.sm; cf* tw = cs.tw; double* red = cs.red;
  uint32_t* tmem_slot = (uint32_t*)((unsigned char*)red + 1000);
  float* Ib = (float*)(cs.pf - t) + t;                        // I (then w) of register r: Ib[r * T]   (thread-private)
  cf* ryS = cs.hyS;                                                 // ry, then rx, of the current position (2 NF entries)
  cs.fill_tables(t);
  if (wp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(tmem_slot)), "n"(TCOLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tb = *tmem_slot + ((uint32_t)((wp & 3) * 32) << 16) + (uint32_t)((wp >> 2) * 128);
  const uint32_t tbT = tb, tbG = tb + 64;                           // columns [0, 64): T ; [64, 128): sum_k gT_k
  const int onx = P.onx;
  const float inv_n = 1.0f / (float)NF;
  cf v[32];
  for (int jl = blockIdx.x; jl < P.jc; jl += gridDim.x) {
    const int jb = P.j0 + jl, row = P.w.rows[jb];
    const int r0y = P.w.r0[2 * jb], r0x = P.w.r0[2 * jb + 1];
    const float4* ob2 = P.w.O2 + ((size_t)r0y * onx + r0x) + (size_t)F::pix_y(0, t, 0) * onx + F::pix_x(0, t, 0);
    const cf* rx = P.w.ramps + (size_t)jb * 2 * NF;
    const cf* ry = rx + NF;
    __syncthreads();                                                // the previous position's readers of ryS / red are done
    if (jl == (int)blockIdx.x) {                                    // first position of this CTA: nobody has prefetched P~_0 yet
      const float4* src = (const float4*)P.w.Pt + t;
#pragma unroll
      for (int p = 0; p < 16; ++p) cp_async16(cs.xs + p * 32, src + p * T);
      cp_async_commit();
    }
    if (t < NF) { ryS[t] = ry[t]; ryS[NF + t] = rx[t]; }            // both shift ramps of the position (read 2M times below)
    for (int b = t * 128; b < F::NNF * 4; b += T * 128)             // this position's measured pattern: DRAM -> L2 now
      l2_prefetch_line((const char*)(P.intensity + (size_t)row * F::NNF) + b);
#pragma unroll
    for (int c = 0; c < 4; ++c) {                                   // H3: the patch, once per position, parked in tensor memory
      cf tt[8];
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const float4 q = ld_nc16(ob2 + F::patch_off(8 * c + 2 * e, onx));
        tt[2 * e] = make_float2(q.x, q.y); tt[2 * e + 1] = make_float2(q.z, q.w);
      }
      tmem_st16(tbT + 16 * c, tt);
    }
    tmem_wait_st();
    cf wxv[F::NXV];
    __syncthreads();                                                // ryS visible
    // One loop over the 2M half steps (pass 1: modes 0..M-1 forward, pass 2: modes 0..M-1 adjoint) so that the kernel holds ONE
    // inverse and ONE forward transform body: with four inlined transforms (~130 KB of code) the loop did not fit the
    // instruction cache and ran three times slower.
#pragma unroll 1
    for (int hs = 0; hs < 2 * P.M; ++hs) {
      const bool fwd_pass = hs < P.M;
      const int k = fwd_pass ? hs : hs - P.M;
      const size_t sk = ((size_t)blockIdx.x * P.M + k) * NNS;       // the CTA's scratch field of mode k: the same lines for every position
                                                                    // the CTA takes, so that they stay in L2 instead of streaming to HBM
      if (hs == P.M) {
        // ---------------- H8: loss and detector weight (float32 per pixel in cancellation-free form, fp64 sum)
        double acc[1] = {0.0};
        const float* Ie = P.intensity + (size_t)row * F::NNF;
        float ls = 0.f, lc = 0.f;                                   // the thread's 32 terms: compensated float32 sum (fp64 conversions
                                                                    // and adds are what made this loop cost 35 k cycles), then fp64
        // Four rounds of eight pixels, NOT unrolled across the rounds: run once per position, the fully unrolled loop (3 loss kinds
        // x 32 pixels, ~3500 instructions = 56 KB) pushed the half-step loop out of the instruction cache (ncu: stall_no_inst was
        // the kernel's first stall reason).  The pattern is in L2 (prefetched at the start of the position).
        float cur[8], nxt[8];                                       // the next round's pattern values are in flight during this one
#pragma unroll
        for (int e = 0; e < 8; ++e) cur[e] = __ldg(Ie + F::fq_y(0, t, e) * NF + F::fq_x(0, t, e));
#pragma unroll 1
        for (int r0 = 0; r0 < 32; r0 += 8) {
          const int rn = r0 + 8 < 32 ? r0 + 8 : r0;                 // (the last round re-reads its own values: no branch)
#pragma unroll
          for (int e = 0; e < 8; ++e) nxt[e] = __ldg(Ie + F::fq_y(0, t, rn + e) * NF + F::fq_x(0, t, rn + e));
#pragma unroll
          for (int e = 0; e < 8; ++e) {
            float l, w;
            pixel_loss_f32(P.loss, Ib[(r0 + e) * T], cur[e], P.eps, P.loss_c, l, w);
            const float y = l - lc, s2 = ls + y;
            lc = (s2 - ls) - y; ls = s2;
            Ib[(r0 + e) * T] = w;
          }
#pragma unroll
          for (int e = 0; e < 8; ++e) cur[e] = nxt[e];
        }
        acc[0] = (double)ls - (double)lc;
        block_sum<G::T, 1>(acc, red);
        if (t == 0) {
          P.w.loss_pp[jb] = acc[0];
          if (!(acc[0] == acc[0]) || fabs(acc[0]) > 1e300) atomicOr(P.w.status, kStatusNonfinite);
        }
      }
      {   // Fourier-side start: H2  R .* P~_k / N^2   or   H9  g~ = w .* psi~_k / N ; the source field (P~_k, or psi~_k from the
          // scratch) was asked into the warp's idle X1 region at the end of the previous half step
        if (fwd_pass) load_xv<G>(wxv, ryS + NF, t, 1.0f / (float)F::NNF);
        cp_async_wait_all();
#pragma unroll
        for (int p = 0; p < 16; ++p) {
          const float4 q = cs.xs[p * 32];
          if (fwd_pass) {
            v[2 * p] = cmul(make_float2(q.x, q.y), cmul(wxv[0], ryS[F::fq_y(0, t, 2 * p)]));
            v[2 * p + 1] = cmul(make_float2(q.z, q.w), cmul(wxv[0], ryS[F::fq_y(0, t, 2 * p + 1)]));
          } else {
            const float w0 = Ib[(2 * p) * T] * inv_n, w1 = Ib[(2 * p + 1) * T] * inv_n;
            v[2 * p] = make_float2(q.x * w0, q.y * w0);
            v[2 * p + 1] = make_float2(q.z * w1, q.w * w1);
          }
        }
      }
      __syncthreads();                                              // every warp has read its source slots: the inverse transform's
                                                                    // CTA-wide exchange may now write into any warp's region
      Fft<G>::inv_head(v, sm, cs.tw2, t, 0u);
      if (!fwd_pass) {   // Psi_k back from the scratch into the warp's idle X1 region (16 slots of 16 B per lane) while phase 1 runs
        const float4* st = (const float4*)(P.w.stash + sk) + t;
#pragma unroll
        for (int p = 0; p < 16; ++p) cp_async16(cs.xs + p * 32, st + p * T);
      }
      cp_async_commit();
      L::phase1_inv(v, tw, t);                                      // Psi_k   or   gPhi_k   (R-layout)
      cp_async_wait_all();
      float4* stw = (float4*)(P.w.stash + sk) + t;
#pragma unroll
      for (int c = 0; c < 8; ++c) {                                 // 8-column tensor-memory accesses (4 complex): see tmem_swap_field
        cf tt[4], ga[4];
        tmem_ld8(tbT + 8 * c, tt);
        if (fwd_pass) {                                             // keep Psi_k for pass 2 ; H4: Phi = Psi_k .* T
#pragma unroll
          for (int e = 0; e < 2; ++e) {
            const int p = 2 * c + e;
            stw[p * T] = make_float4(v[2 * p].x, v[2 * p].y, v[2 * p + 1].x, v[2 * p + 1].y);
            v[2 * p] = cmul(v[2 * p], tt[2 * e]);
            v[2 * p + 1] = cmul(v[2 * p + 1], tt[2 * e + 1]);
          }
        } else {                                                    // H10: gT += conj(Psi_k) gPhi ; gPsi = conj(T) gPhi
          if (k > 0) tmem_ld8(tbG + 8 * c, ga);
#pragma unroll
          for (int e = 0; e < 2; ++e) {
            const int p = 2 * c + e;
            const float4 ps = cs.xs[p * 32];
            const cf g0 = cmulc(v[2 * p], make_float2(ps.x, ps.y)), g1 = cmulc(v[2 * p + 1], make_float2(ps.z, ps.w));
            ga[2 * e] = k > 0 ? cadd(ga[2 * e], g0) : g0;
            ga[2 * e + 1] = k > 0 ? cadd(ga[2 * e + 1], g1) : g1;
            v[2 * p] = cmulc(v[2 * p], tt[2 * e]);
            v[2 * p + 1] = cmulc(v[2 * p + 1], tt[2 * e + 1]);
          }
          if (k + 1 < P.M) tmem_st8(tbG + 8 * c, ga);
          else {                                                    // last mode: the sum over the modes goes to the staging buffer
            float4* gt = (float4*)(P.w.gTpart + (size_t)jl * NNS) + t;
#pragma unroll
            for (int e = 0; e < 2; ++e) __stcs(gt + (2 * c + e) * T, make_float4(ga[2 * e].x, ga[2 * e].y, ga[2 * e + 1].x, ga[2 * e + 1].y));
          }
        }
      }
      tmem_wait_st();
      Fft<G>::fwd(v, sm, tw, cs.tw2, t, 0u);                        // F(Phi)   or   G~ = F(gPsi)
      // the next half step's source field -> the warp's X1 region (free until that half step's inverse transform): P~ of the next
      // mode, psi~ of the first / next mode from the scratch, or P~_0 again for the CTA's next position.  Issued before the tail
      // below so that the copy overlaps it — except when the field is psi~_0 and this half step is about to store it (M = 1)
      const int hn = hs + 1;
      auto prefetch_next = [&]() {
        const cf* nsrc = hn < P.M ? P.w.Pt + (size_t)hn * NNS : hn < 2 * P.M ? P.w.psit + ((size_t)blockIdx.x * P.M + (hn - P.M)) * NNS : P.w.Pt;
        const float4* src = (const float4*)nsrc + t;
#pragma unroll
        for (int p = 0; p < 16; ++p) cp_async16(cs.xs + p * 32, src + p * T);
        cp_async_commit();
        // and Psi of the next adjoint half step towards L2 (its cp.async is issued only after that half step's inverse-transform head)
        if (hn >= P.M && hn < 2 * P.M)
          for (int b = t * 128; b < NNS * 8; b += T * 128) l2_prefetch_line((const char*)(P.w.stash + ((size_t)blockIdx.x * P.M + (hn - P.M)) * NNS) + b);
      };
      if (hn != P.M) prefetch_next();
      if (fwd_pass) {
        float4* out = (float4*)(P.w.psit + sk) + t;                 // H6: psi~_k = F(Phi) / N ; H7: I += |psi~_k|^2
#pragma unroll
        for (int p = 0; p < 16; ++p) {
          const float4 q = make_float4(v[2 * p].x * inv_n, v[2 * p].y * inv_n, v[2 * p + 1].x * inv_n, v[2 * p + 1].y * inv_n);
          out[p * T] = q;
          const float i0 = fmaf(q.x, q.x, q.y * q.y), i1 = fmaf(q.z, q.z, q.w * q.w);
          Ib[(2 * p) * T] = k == 0 ? i0 : Ib[(2 * p) * T] + i0;
          Ib[(2 * p + 1) * T] = k == 0 ? i1 : Ib[(2 * p + 1) * T] + i1;
        }
        if (hn == P.M) prefetch_next();                             // psi~_0, after this thread's own store of it (M = 1)
      } else {
        // H12: probe partial conj(R) .* G~ ;  H13: (4 pi / N^2) sum_q f_a Im(conj(G~) R P~)
        const float4* pt4 = (const float4*)(P.w.Pt + (size_t)k * NNS) + t;
        // probe partial: ONE plane per (CTA, mode), the CTA's positions added in the order it takes them (float32, one adder per
        // address, program order: deterministic) — 1/7 of the planes at config 2 for the probe reduction to read
        float4* gp4 = (float4*)(P.w.Gpart + ((size_t)blockIdx.x * P.M + k) * NNS) + t;
        const bool first_pos = jl == (int)blockIdx.x;
        load_xv<G>(wxv, ryS + NF, t, 1.0f);
        float sy = 0.f, sx = 0.f;
        const float fx = (float)signed_freq(F::fq_x(0, t, 0), NF) / (float)NF;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          float4 q[4];                                              // P~ of four register pairs in flight before their use
#pragma unroll
          for (int e = 0; e < 4; ++e) q[e] = want_pos ? __ldg(pt4 + (4 * c + e) * T) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const int p = 4 * c + e;
            const int qy0 = F::fq_y(0, t, 2 * p), qy1 = F::fq_y(0, t, 2 * p + 1);
            const cf R0 = cmul(wxv[0], ryS[qy0]), R1 = cmul(wxv[0], ryS[qy1]);
            const cf g0 = cmulc(v[2 * p], R0), g1 = cmulc(v[2 * p + 1], R1);
            if (first_pos) gp4[p * T] = make_float4(g0.x, g0.y, g1.x, g1.y);
            else asm volatile("red.global.add.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(gp4 + p * T), "f"(g0.x), "f"(g0.y), "f"(g1.x), "f"(g1.y) : "memory");
            if (want_pos) {
              const cf z0 = cmulc(cmul(R0, make_float2(q[e].x, q[e].y)), v[2 * p]), z1 = cmulc(cmul(R1, make_float2(q[e].z, q[e].w)), v[2 * p + 1]);
              sy = fmaf((float)signed_freq(qy0, NF) * (1.0f / (float)NF), z0.y, sy); sx = fmaf(fx, z0.y, sx);
              sy = fmaf((float)signed_freq(qy1, NF) * (1.0f / (float)NF), z1.y, sy); sx = fmaf(fx, z1.y, sx);
            }
          }
        }
        if (want_pos) {
          double acc[2] = {(double)sy, (double)sx};
          block_sum<G::T, 2>(acc, red);
          if (t == 0) {
            const double f = 4.0 * CUDART_PI / ((double)NF * (double)NF);
            P.w.posg_part[((size_t)jb * P.M + k) * 2 + 0] = f * acc[0];
            P.w.posg_part[((size_t)jb * P.M + k) * 2 + 1] = f * acc[1];
          }
        }
      }
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (wp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(*tmem_slot), "n"(TCOLS));
}

// ------------------------------------------------------------------------------------------------
// ePIE normalisations: tmax[jl][i] = max over the window of |O_i|^2 ; psimax[block] = max |Psi|^2 of
// one 16384-element block of the stash (one per (pair, slice, rank); the backward kernel takes the max over the ranks).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float block_max256(float v, float* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  float m = red[0];
  for (int w = 1; w < 8; ++w) m = fmaxf(m, red[w]);
  return m;
}
__global__ void __launch_bounds__(256) k_patch_max(KP P) {
  __shared__ float red[8];
  const int jl = blockIdx.x / P.S, i = blockIdx.x - jl * P.S, jb = P.j0 + jl, N = P.N;
  const cf* o = P.object + ((size_t)i * P.ony + P.w.r0[2 * jb]) * P.onx + P.w.r0[2 * jb + 1];
  float m = 0.f;
  for (int e = threadIdx.x; e < N * N; e += 256) { const cf z = o[(size_t)(e / N) * P.onx + (e % N)]; m = fmaxf(m, fmaf(z.x, z.x, z.y * z.y)); }
  m = block_max256(m, red);
  if (threadIdx.x == 0) P.w.tmax[(size_t)jl * P.S + i] = m;
}
__global__ void __launch_bounds__(256) k_stash_max(const cf* stash, float* out, int n_per_block) {
  __shared__ float red[8];
  const cf* s = stash + (size_t)blockIdx.x * n_per_block;
  float m = 0.f;
  for (int e = threadIdx.x; e < n_per_block; e += 256) { const cf z = s[e]; m = fmaxf(m, fmaf(z.x, z.x, z.y * z.y)); }
  m = block_max256(m, red);
  if (threadIdx.x == 0) out[blockIdx.x] = m;
}

// ------------------------------------------------------------------------------------------------
// Bilinear mode (reading R1, secondary): H3 as a pre-pass.  Tb[jl][i][y][x] = sum_d w_d O_i[i0 + (y,x) + d],
// w_d = (d_y ? f_y : 1 - f_y)(d_x ? f_x : 1 - f_x); the chain kernels then read these patches instead of the
// object window.  One block per (position of the chunk, slice).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_bilinear_patches(KP P, int D) {   // D: distance of a pixel's partner (as k_pair_object)
  const int jl = blockIdx.x / P.S, i = blockIdx.x - jl * P.S, jb = P.j0 + jl, N = P.N;
  const int i0y = P.w.r0[2 * jb], i0x = P.w.r0[2 * jb + 1];
  const float fy = P.w.delta[2 * jb], fx = P.w.delta[2 * jb + 1];
  const float w00 = (1.f - fy) * (1.f - fx), w01 = (1.f - fy) * fx, w10 = fy * (1.f - fx), w11 = fy * fx;
  const cf* o = P.object + ((size_t)i * P.ony + i0y) * P.onx + i0x;
  float4* out = P.w.Tb + ((size_t)jl * P.S + i) * N * N;
  auto sample = [&](int y, int x) {
    const cf a = o[(size_t)y * P.onx + x], b = o[(size_t)y * P.onx + x + 1], c = o[(size_t)(y + 1) * P.onx + x], d = o[(size_t)(y + 1) * P.onx + x + 1];
    return make_float2(w00 * a.x + w01 * b.x + w10 * c.x + w11 * d.x, w00 * a.y + w01 * b.y + w10 * c.y + w11 * d.y);
  };
  for (int e = threadIdx.x; e < N * N; e += 256) {
    const int y = e / N, x = e - y * N;
    const cf u = sample(y, x), w = x + D < N ? sample(y, x + D) : make_float2(0.f, 0.f);
    out[e] = make_float4(u.x, u.y, w.x, w.y);
  }
}

// Bilinear mode, H13: dL/df_a = 2 Re sum_i sum_r conj(gT_i[r]) dT_i[r]/df_a with gT summed over the modes in fixed
// order; dT/df_y = sum_dx w_dx (O[y+1, x+dx] - O[y, x+dx]), dT/df_x likewise.  One block per position of the chunk.
template <class G>
__global__ void __launch_bounds__(256) k_pos_bilinear(KP P, int cl) {
  typedef FL<G> F;
  constexpr int N = F::NF, NN = F::NNF;
  __shared__ double red[(256 / 32) * 2];
  const int jl = blockIdx.x, jb = P.j0 + jl;
  const int i0y = P.w.r0[2 * jb], i0x = P.w.r0[2 * jb + 1];
  const double fy = (double)P.w.delta[2 * jb], fx = (double)P.w.delta[2 * jb + 1];
  double acc[2] = {0.0, 0.0};
  for (int i = 0; i < P.S; ++i) {
    const cf* o = P.object + ((size_t)i * P.ony + i0y) * P.onx + i0x;
    for (int e = threadIdx.x; e < NN; e += 256) {
      const int y = e / N, x = e - y * N;
      const size_t base = ((size_t)jl * P.Mg * P.S + i) * NN + F::r_native_of(y, x);
      double gr = 0.0, gi = 0.0;
      for (int k = 0; k < P.Mg; ++k) { const cf g = P.w.gTpart[base + (size_t)k * P.S * NN]; gr += (double)g.x; gi += (double)g.y; }
      const cf a = o[(size_t)y * P.onx + x], b = o[(size_t)y * P.onx + x + 1], c = o[(size_t)(y + 1) * P.onx + x], d = o[(size_t)(y + 1) * P.onx + x + 1];
      const double tyr = (1.0 - fx) * ((double)c.x - a.x) + fx * ((double)d.x - b.x), tyi = (1.0 - fx) * ((double)c.y - a.y) + fx * ((double)d.y - b.y);
      const double txr = (1.0 - fy) * ((double)b.x - a.x) + fy * ((double)d.x - c.x), txi = (1.0 - fy) * ((double)b.y - a.y) + fy * ((double)d.y - c.y);
      acc[0] += 2.0 * (gr * tyr + gi * tyi);                     // 2 Re(conj(g) dT)
      acc[1] += 2.0 * (gr * txr + gi * txi);
    }
  }
  block_sum<256, 2>(acc, red);
  if (threadIdx.x == 0) {
    const int MU = P.M * cl;
    for (int u = 0; u < MU; ++u) {                               // k_finalize sums the MU per-(mode, rank) slots
      P.w.posg_part[((size_t)jb * MU + u) * 2 + 0] = u == 0 ? acc[0] : 0.0;
      P.w.posg_part[((size_t)jb * MU + u) * 2 + 1] = u == 0 ? acc[1] : 0.0;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// H11: deterministic object-gradient scatter-add as an owner-computes gather.  Block = 64 x 4 object pixels of
// one slice; each pixel sums, in fixed (j ascending, k ascending) order, the patch-gradient entries that
// land on it, in fp64, then adds the chunk total to gO once.  Optionally the illumination map (O12).
// ------------------------------------------------------------------------------------------------
#ifndef GATHER_TW
#define GATHER_TW 64     // tile width in object pixels (256 threads per block)
#endif
template <class G, bool ILLUM, bool BILIN>
__global__ void __launch_bounds__(256, ILLUM ? 8 : 0) k_gather_object(KP P, cf* gO, float* illum) {
  typedef FL<G> F;
  constexpr int N = F::NF, NN = F::NNF, NR = BILIN ? N + 1 : N;   // bilinear mode: a window deposits on N + 1 pixels per axis
  __shared__ int2 sr0[256];
  __shared__ float2 sfr[BILIN ? 256 : 1];
  const int i = blockIdx.z;
  constexpr int TW_ = GATHER_TW, TH_ = 256 / GATHER_TW;
  const int ox0 = blockIdx.x * TW_, oy0 = blockIdx.y * TH_;
  const int ox = ox0 + threadIdx.x, oy = oy0 + threadIdx.y;
  const int tid = threadIdx.y * TW_ + threadIdx.x;
  double ar = 0.0, ai = 0.0, al = 0.0;
  for (int jbase = 0; jbase < P.jc; jbase += 256) {
    const int cnt = min(256, P.jc - jbase);
    if (tid < cnt) {
      sr0[tid] = make_int2(P.w.r0[2 * (P.j0 + jbase + tid) + 1], P.w.r0[2 * (P.j0 + jbase + tid)]);  // (x, y)
      if (BILIN) sfr[tid] = make_float2(P.w.delta[2 * (P.j0 + jbase + tid) + 1], P.w.delta[2 * (P.j0 + jbase + tid)]);  // (fx, fy)
    }
    __syncthreads();
    // which windows reach this tile: every lane tests one window of a group of 32 (the test is block-uniform, so all
    // warps get the same mask), then the warp walks the set bits in ascending order — the summation order is unchanged
    for (int grp = 0; grp < cnt; grp += 32) {
      bool hit = false;
      if (grp + (tid & 31) < cnt) {
        const int2 q = sr0[grp + (tid & 31)];
        hit = !(q.x > ox0 + TW_ - 1 || q.x + NR <= ox0 || q.y > oy0 + TH_ - 1 || q.y + NR <= oy0);
      }
      unsigned hits = __ballot_sync(0xffffffffu, hit);
      while (hits) {
      const int jj = grp + __ffs(hits) - 1;
      hits &= hits - 1;
      const int2 r0 = sr0[jj];
      const int px = ox - r0.x, py = oy - r0.y;
      if (BILIN) {
        // adjoint of the four-tap sampling: pixel o collects w_d gT[o - i0 - d] (the same weights)
        if (px >= 0 && px <= N && py >= 0 && py <= N) {
          const double fx = (double)sfr[jj].x, fy = (double)sfr[jj].y;
#pragma unroll
          for (int d = 0; d < 4; ++d) {
            const int dy = d >> 1, dx = d & 1, ry = py - dy, rx = px - dx;
            if (ry < 0 || ry >= N || rx < 0 || rx >= N) continue;
            const double wgt = (dy ? fy : 1.0 - fy) * (dx ? fx : 1.0 - fx);
            const int nat = F::r_native_of(ry, rx);
            const size_t base = ((size_t)(jbase + jj) * P.Mg * P.S + i) * NN + nat;
            double sr = 0.0, si = 0.0, sl = 0.0;
            for (int k = 0; k < P.Mg; ++k) { const cf g = P.w.gTpart[base + (size_t)k * P.S * NN]; sr += (double)g.x; si += (double)g.y; }
            if (ILLUM) {
              const size_t sb = ((size_t)(jbase + jj) * P.M * P.S + i) * NN + nat, sbs = ((size_t)(jbase + jj) * P.Mi * P.S + i) * NN + nat;
              if (P.w.ilpart) for (int k = 0; k < P.Mi; ++k) sl += (double)P.w.ilpart[sbs + (size_t)k * P.S * NN];
              else for (int k = 0; k < P.M; ++k) { const cf q = P.w.stash[sb + (size_t)k * P.S * NN]; sl += (double)q.x * q.x + (double)q.y * q.y; }
            }
            ar += wgt * sr; ai += wgt * si; al += wgt * sl;
          }
        }
      } else if (px >= 0 && px < N && py >= 0 && py < N) {
        const int idx = F::r_native_of(py, px);
        const size_t base = ((size_t)(jbase + jj) * P.Mg * P.S + i) * NN + idx;
        for (int k = 0; k < P.Mg; ++k) { const cf g = P.w.gTpart[base + (size_t)k * P.S * NN]; ar += (double)g.x; ai += (double)g.y; }
        if (ILLUM) {
          const size_t sb = ((size_t)(jbase + jj) * P.M * P.S + i) * NN + idx, sbs = ((size_t)(jbase + jj) * P.Mi * P.S + i) * NN + idx;
          if (P.w.ilpart) for (int k = 0; k < P.Mi; ++k) al += (double)P.w.ilpart[sbs + (size_t)k * P.S * NN];   // staged by the backward kernel
          else for (int k = 0; k < P.M; ++k) { const cf s = P.w.stash[sb + (size_t)k * P.S * NN]; al += (double)s.x * s.x + (double)s.y * s.y; }
        }
      }
      }
    }
    __syncthreads();
  }
  if (ox < P.onx && oy < P.ony) {
    const size_t o = ((size_t)i * P.ony + oy) * P.onx + ox;
    cf cur = gO[o];
    gO[o] = make_float2((float)((double)cur.x + ar), (float)((double)cur.y + ai));
    if (ILLUM) illum[o] = (float)((double)illum[o] + al);
  }
}

// The same gather with the chunk's windows split over the eight warps of a block (used when the object has few tiles): a block owns
// 32 object pixels of one row; warp w walks the window groups g = w, w + 8, ... (32 windows per group, one window test per lane,
// ballot), every lane accumulates its pixel over the hits in ascending order, and the eight partial sums are added in warp order
// 0..7: still a fixed order, with eight times the loads in flight per pixel.
template <class G, bool ILLUM, bool BILIN>
__global__ void __launch_bounds__(256) k_gather_object_w(KP P, cf* gO, float* illum) {
  typedef FL<G> F;
  constexpr int N = F::NF, NN = F::NNF, NR = BILIN ? N + 1 : N;
  __shared__ double part[8][3][32];
  const int i = blockIdx.z, lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int ox0 = blockIdx.x * 32, oy = blockIdx.y, ox = ox0 + lane;
  double ar = 0.0, ai = 0.0, al = 0.0;
  for (int grp = w * 32; grp < P.jc; grp += 256) {
    int2 q = make_int2(0, 0);
    bool hit = false;
    if (grp + lane < P.jc) {
      q = make_int2(P.w.r0[2 * (P.j0 + grp + lane) + 1], P.w.r0[2 * (P.j0 + grp + lane)]);   // (x, y)
      hit = !(q.x > ox0 + 31 || q.x + NR <= ox0 || q.y > oy || q.y + NR <= oy);
    }
    unsigned hits = __ballot_sync(0xffffffffu, hit);
    while (hits) {
      const int b = __ffs(hits) - 1, jj = grp + b;
      hits &= hits - 1;
      const int px = ox - __shfl_sync(0xffffffffu, q.x, b), py = oy - __shfl_sync(0xffffffffu, q.y, b);
      if (BILIN) {
        if (px >= 0 && px <= N && py >= 0 && py <= N) {
          const double fx = (double)P.w.delta[2 * (P.j0 + jj) + 1], fy = (double)P.w.delta[2 * (P.j0 + jj)];
#pragma unroll
          for (int d = 0; d < 4; ++d) {
            const int dy = d >> 1, dx = d & 1, ry = py - dy, rx = px - dx;
            if (ry < 0 || ry >= N || rx < 0 || rx >= N) continue;
            const double wgt = (dy ? fy : 1.0 - fy) * (dx ? fx : 1.0 - fx);
            const int nat = F::r_native_of(ry, rx);
            const size_t base = ((size_t)jj * P.Mg * P.S + i) * NN + nat;
            double sr = 0.0, si = 0.0, sl = 0.0;
            for (int k = 0; k < P.Mg; ++k) { const cf g = P.w.gTpart[base + (size_t)k * P.S * NN]; sr += (double)g.x; si += (double)g.y; }
            if (ILLUM) {
              const size_t sb = ((size_t)jj * P.M * P.S + i) * NN + nat, sbs = ((size_t)jj * P.Mi * P.S + i) * NN + nat;
              if (P.w.ilpart) for (int k = 0; k < P.Mi; ++k) sl += (double)P.w.ilpart[sbs + (size_t)k * P.S * NN];
              else for (int k = 0; k < P.M; ++k) { const cf z = P.w.stash[sb + (size_t)k * P.S * NN]; sl += (double)z.x * z.x + (double)z.y * z.y; }
            }
            ar += wgt * sr; ai += wgt * si; al += wgt * sl;
          }
        }
      } else if (px >= 0 && px < N && py >= 0 && py < N) {
        const int idx = F::r_native_of(py, px);
        const size_t base = ((size_t)jj * P.Mg * P.S + i) * NN + idx;
        for (int k = 0; k < P.Mg; ++k) { const cf g = P.w.gTpart[base + (size_t)k * P.S * NN]; ar += (double)g.x; ai += (double)g.y; }
        if (ILLUM) {
          const size_t sb = ((size_t)jj * P.M * P.S + i) * NN + idx, sbs = ((size_t)jj * P.Mi * P.S + i) * NN + idx;
          if (P.w.ilpart) for (int k = 0; k < P.Mi; ++k) al += (double)P.w.ilpart[sbs + (size_t)k * P.S * NN];
          else for (int k = 0; k < P.M; ++k) { const cf z = P.w.stash[sb + (size_t)k * P.S * NN]; al += (double)z.x * z.x + (double)z.y * z.y; }
        }
      }
    }
  }
  part[w][0][lane] = ar; part[w][1][lane] = ai; part[w][2][lane] = al;
  __syncthreads();
  if (w == 0 && ox < P.onx) {
    double sr = 0.0, si = 0.0, sl = 0.0;
#pragma unroll
    for (int ww = 0; ww < 8; ++ww) { sr += part[ww][0][lane]; si += part[ww][1][lane]; sl += part[ww][2][lane]; }
    const size_t o = ((size_t)i * P.ony + oy) * P.onx + ox;
    const cf cur = gO[o];
    gO[o] = make_float2((float)((double)cur.x + sr), (float)((double)cur.y + si));
    if (ILLUM) illum[o] = (float)((double)illum[o] + sl);
  }
}

// ------------------------------------------------------------------------------------------------
// LSQML slice update with per-position step sizes (reading R24).
// k_alpha_pos: alpha_{O,i,j} = numO[j,i] / (denO[j,i] + gamma) from the per-(mode, rank) fp64 partials of the sweep that
// has just run over this chunk (fixed order).  k_gather_willum: W_i[r] += sum_j alpha_{O,i,j} sum_k |Psi_{i,k,j}[r - r0_j]|^2,
// the same owner-computes gather as k_gather_object over the staged |Psi|^2 (fixed (j, k) order, fp64).
// ------------------------------------------------------------------------------------------------
__global__ void k_alpha_pos(KP P, float gamma) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= P.jc * P.S) return;
  const int jl = idx / P.S, i = idx - jl * P.S;
  const double* sp = P.w.step_oi + ((size_t)(P.j0 + jl) * P.S + i) * 6;
  P.w.alpha_ji[idx] = (float)(sp[0] / (sp[1] + (double)gamma));
}
template <class G>
__global__ void __launch_bounds__(256) k_gather_willum(KP P, float* willum) {
  typedef FL<G> F;
  constexpr int N = F::NF, NN = F::NNF, TW_ = GATHER_TW, TH_ = 256 / GATHER_TW;
  __shared__ int2 sr0[256];
  __shared__ float sal[256];
  const int i = blockIdx.z;
  const int ox0 = blockIdx.x * TW_, oy0 = blockIdx.y * TH_;
  const int ox = ox0 + threadIdx.x, oy = oy0 + threadIdx.y;
  const int tid = threadIdx.y * TW_ + threadIdx.x;
  double acc = 0.0;
  for (int jbase = 0; jbase < P.jc; jbase += 256) {
    const int cnt = min(256, P.jc - jbase);
    if (tid < cnt) {
      sr0[tid] = make_int2(P.w.r0[2 * (P.j0 + jbase + tid) + 1], P.w.r0[2 * (P.j0 + jbase + tid)]);  // (x, y)
      sal[tid] = P.w.alpha_ji[(size_t)(jbase + tid) * P.S + i];
    }
    __syncthreads();
    for (int g = 0; g < cnt; g += 32) {                          // as in k_gather_object: ballot over a group of 32 windows
      bool hit = false;
      if (g + (tid & 31) < cnt) {
        const int2 q = sr0[g + (tid & 31)];
        hit = !(q.x > ox0 + TW_ - 1 || q.x + N <= ox0 || q.y > oy0 + TH_ - 1 || q.y + N <= oy0);
      }
      unsigned hits = __ballot_sync(0xffffffffu, hit);
      while (hits) {
        const int jj = g + __ffs(hits) - 1;
        hits &= hits - 1;
        const int2 r0 = sr0[jj];
        const int px = ox - r0.x, py = oy - r0.y;
        if (px >= 0 && px < N && py >= 0 && py < N) {
          const size_t base = ((size_t)(jbase + jj) * P.Mi * P.S + i) * NN + F::r_native_of(py, px);
          double s = 0.0;
          for (int k = 0; k < P.Mi; ++k) s += (double)P.w.ilpart[base + (size_t)k * P.S * NN];      // |Psi_{i,k}|^2 staged by the backward kernel
          acc += (double)sal[jj] * s;
        }
      }
    }
    __syncthreads();
  }
  if (ox < P.onx && oy < P.ony) {
    const size_t o = ((size_t)i * P.ony + oy) * P.onx + ox;
    willum[o] = (float)((double)willum[o] + acc);
  }
}

// ------------------------------------------------------------------------------------------------
// LSQML probe preconditioner (R25): objtrans[r] = sum_j prod_i |O_i[r0_j + r]|^2, one thread per window pixel,
// positions in fixed order, fp64.  The position split is the fp32 arithmetic of k_setup_pos (R2), clamped + flagged (R4).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_objtrans(KP P, float* out, int accumulate) {
  __shared__ int2 sr0[256];
  const int N = P.N, e = blockIdx.x * 256 + threadIdx.x, y = e / N, x = e - y * N;
  double acc = 0.0;
  for (int jbase = 0; jbase < P.J; jbase += 256) {
    const int cnt = min(256, P.J - jbase);
    if ((int)threadIdx.x < cnt) {
      const int jb = jbase + threadIdx.x;
      int row = P.batch_idx ? P.batch_idx[jb] : jb;
      if (row < 0 || row >= P.Jtot) { atomicOr(P.w.status, kStatusOOB); row = row < 0 ? 0 : P.Jtot - 1; }
      int r0[2];
#pragma unroll
      for (int a = 0; a < 2; ++a) {
        const float c = __fsub_rn(__fdiv_rn(P.positions[2 * row + a], P.px), (float)(N / 2));
        int r = (int)floorf(__fadd_rn(c, 0.5f));
        const int lim = (a == 0 ? P.ony : P.onx) - N;
        if (r < 0 || r > lim) { atomicOr(P.w.status, kStatusOOB); r = r < 0 ? 0 : lim; }
        r0[a] = r;
      }
      sr0[threadIdx.x] = make_int2(r0[1], r0[0]);
    }
    __syncthreads();
    for (int jj = 0; jj < cnt; ++jj) {
      const cf* o = P.object + ((size_t)(sr0[jj].y + y)) * P.onx + sr0[jj].x + x;
      float tr = 1.0f;
      for (int i = 0; i < P.S; ++i) { const cf z = o[(size_t)i * P.ony * P.onx]; tr *= fmaf(z.x, z.x, z.y * z.y); }
      acc += (double)tr;
    }
    __syncthreads();
  }
  out[e] = (float)((accumulate ? (double)out[e] : 0.0) + acc);
}

// H12: gP~_k[q] += sum_j (chunk) conj(R_j) G~_{k,j}[q], fixed order, fp64, in two stages so that the chunk's positions are summed
// by kReduceZ blocks side by side: stage 1 sums a contiguous range of positions into part[z][k][q], stage 2 adds the kReduceZ
// partial sums in order z = 0, 1, ... to the accumulator.
__global__ void k_reduce_probe(KP P, double2* part) {
  const int NN = P.N * P.N;
  const int e = blockIdx.x * blockDim.x + threadIdx.x, k = blockIdx.y, z = blockIdx.z;
  if (e >= NN) return;
  const int per = (P.jc + kReduceZ - 1) / kReduceZ, lo = z * per, hi = min(P.jc, lo + per);
  double ar = 0.0, ai = 0.0;
#pragma unroll 8                                                    // eight loads in flight, the additions in the same order (0.95 -> 0.71 ms at config 3)
  for (int jl = lo; jl < hi; ++jl) {
    const cf g = P.w.Gpart[(size_t)(jl * P.M + k) * NN + e];
    ar += (double)g.x; ai += (double)g.y;
  }
  part[((size_t)z * P.M + k) * NN + e] = make_double2(ar, ai);
}
__global__ void k_reduce_probe2(KP P, const double2* part) {
  const int NN = P.N * P.N;
  const int e = blockIdx.x * blockDim.x + threadIdx.x, k = blockIdx.y;
  if (e >= NN) return;
  double2 a = P.w.gPt_acc[(size_t)k * NN + e];
  for (int z = 0; z < kReduceZ; ++z) { const double2 q = part[((size_t)z * P.M + k) * NN + e]; a.x += q.x; a.y += q.y; }
  P.w.gPt_acc[(size_t)k * NN + e] = a;
}

// loss total (fixed-order fp64), position gradients (sum over modes, / px), step-term sums over modes
// (cl = CTAs per field: every per-(position, mode) partial exists once per cluster rank)
__global__ void k_finalize(KP P, int cl, double* loss, int accumulate, float* loss_per_pos, float* grad_pos, float* step_terms) {
  __shared__ double red[1024 / 32];
  const int t = threadIdx.x, MU = P.M * cl;
  if (loss || loss_per_pos) {
    double acc[1] = {0.0};
    for (int j = t; j < P.J; j += 1024) {
      double lj = 0.0;
      for (int c = 0; c < cl; ++c) lj += P.w.loss_pp[(size_t)j * cl + c];
      if (loss_per_pos) loss_per_pos[j] = (float)lj;
      acc[0] += lj;
    }
    block_sum<1024, 1>(acc, red);
    if (t == 0 && loss) *loss = (accumulate ? *loss : 0.0) + acc[0];
  }
  if (grad_pos)
    for (int j = t; j < P.J; j += 1024) {
      double sy = 0.0, sx = 0.0;
      for (int k = 0; k < MU; ++k) { sy += P.w.posg_part[((size_t)j * MU + k) * 2]; sx += P.w.posg_part[((size_t)j * MU + k) * 2 + 1]; }
      grad_pos[2 * j] = (float)(sy / (double)P.px);
      grad_pos[2 * j + 1] = (float)(sx / (double)P.px);
    }
  if (step_terms) {
    // object terms per (position, slice); probe terms summed over the modes (and ranks); position terms likewise, or (bilinear
    // mode, where they come through the patch) summed over the slices
    const int W = 2 * P.S + 6;
    for (int idx = t; idx < P.J * W; idx += 1024) {
      const int j = idx / W, c = idx - j * W;
      double s = 0.0;
      if (c < 2 * P.S) s = P.w.step_oi[((size_t)j * P.S + (c >> 1)) * 6 + (c & 1)];
      else if (c >= 2 * P.S + 2 && P.bilinear) for (int i = 0; i < P.S; ++i) s += P.w.step_oi[((size_t)j * P.S + i) * 6 + (c - 2 * P.S)];
      else for (int k = 0; k < MU; ++k) s += P.w.step_pp[((size_t)j * MU + k) * 6 + (c - 2 * P.S)];
      step_terms[idx] = (float)s;
    }
  }
}


// O13: dOhat = -gO / (illum_prev + delta_O)
__global__ void k_dohat(const cf* gO, const float* illum_prev, float delta_o, cf* out, size_t n) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const float d = -1.0f / (illum_prev[i] + delta_o);
  out[i] = make_float2(gO[i].x * d, gO[i].y * d);
}

// ------------------------------------------------------------------------------------------------
// H15 update kernels
// ------------------------------------------------------------------------------------------------
__global__ void k_axpy(float* z, const float* g, float a, size_t n) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) z[i] = fmaf(a, g[i], z[i]);
}
// (rows outside [0, n_rows) are skipped; the gradient call that produced g has already raised PT_ERR_OUT_OF_BOUNDS for them.
//  A batch must not name a row twice: the two updates would race.)
// the whole SGD step in one launch: blocks [0, bo) the object, [bo, bo + bp) the probe, the rest the positions (same arithmetic
// per element as k_axpy; positions: pos[row] -= lr g[j])
__global__ void k_sgd(float* obj, const float* gO, float ao, size_t no, unsigned bo, float* pr, const float* gP, float ap, size_t np, unsigned bp,
                      float* pos, const float* gX, const int32_t* idx, float lr, int J, int n_rows) {
  if (blockIdx.x < bo) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < no) obj[i] = fmaf(ao, gO[i], obj[i]);
  } else if (blockIdx.x < bo + bp) {
    const size_t i = (size_t)(blockIdx.x - bo) * blockDim.x + threadIdx.x;
    if (i < np) pr[i] = fmaf(ap, gP[i], pr[i]);
  } else {
    const int j = (int)(blockIdx.x - bo - bp) * blockDim.x + threadIdx.x;
    if (j >= J) return;
    const int row = idx ? idx[j] : j;
    if (row < 0 || row >= n_rows) return;
    pos[2 * row] -= lr * gX[2 * j]; pos[2 * row + 1] -= lr * gX[2 * j + 1];
  }
}
// alpha[c] = sum_j num / (sum_j den + gamma) for c = 0..S (S object slices, then the probe); one block per c
__global__ void k_lsqml_alpha(const float* step_terms, int J, int S, float gamma, float* alpha) {
  __shared__ double red[(256 / 32) * 2];
  const int c = blockIdx.x, W = 2 * S + 6;
  double acc[2] = {0.0, 0.0};
  for (int j = threadIdx.x; j < J; j += 256) { acc[0] += step_terms[(size_t)j * W + 2 * c]; acc[1] += step_terms[(size_t)j * W + 2 * c + 1]; }
  block_sum<256, 2>(acc, red);
  if (threadIdx.x == 0) alpha[c] = (float)(acc[0] / (acc[1] + (double)gamma));
}
__global__ void k_lsqml_object(cf* O, const cf* gO, const float* illum_prev, const float* alpha, float beta, float delta_o,
                               size_t slice_elems, size_t n) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const float a = beta * alpha[i / slice_elems] * (-1.0f / (illum_prev[i] + delta_o));
  O[i] = make_float2(fmaf(a, gO[i].x, O[i].x), fmaf(a, gO[i].y, O[i].y));
}
// PAPER.md:225 as printed (R24): O_i += beta dOhat_i W_i / I_i where I_i > 0, dOhat = -gO / (illum_prev + delta_O)
__global__ void k_lsqml_object_weighted(cf* O, const cf* gO, const float* illum_prev, const float* illum_batch, const float* willum,
                                        float beta, float delta_o, size_t n) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const float ib = illum_batch[i];
  if (!(ib > 0.f)) return;
  const float a = beta * (willum[i] / ib) * (-1.0f / (illum_prev[i] + delta_o));
  O[i] = make_float2(fmaf(a, gO[i].x, O[i].x), fmaf(a, gO[i].y, O[i].y));
}
__global__ void k_lsqml_probe(cf* Pr, const cf* gP, const float* alpha, int S, float beta, float delta_p, const float* precond, size_t NN, size_t n) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const float a = beta * alpha[S] * (-1.0f / ((precond ? precond[i % NN] : 1.0f) + delta_p));
  Pr[i] = make_float2(fmaf(a, gP[i].x, Pr[i].x), fmaf(a, gP[i].y, Pr[i].y));
}
__global__ void k_lsqml_pos(float* pos, const float* step_terms, const int32_t* idx, int J, int S, float px, float gamma, int n_rows) {
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= J) return;
  const int W = 2 * S + 6; int row = idx ? idx[j] : j;
  if (row < 0 || row >= n_rows) return;
  const float* s = step_terms + (size_t)j * W + 2 * S + 2;
  pos[2 * row] += px * s[0] / (s[1] + gamma);
  pos[2 * row + 1] += px * s[2] / (s[3] + gamma);
}

// ------------------------------------------------------------------------------------------------
// launch accounting + optional per-kernel timing (ptycho_profile_*): when enabled, one CUDA event is recorded on
// the launching stream after every kernel (and one at the start of each public call); a stream runs its work in
// order, so the time between consecutive events is that kernel's duration as seen on the device.
// ------------------------------------------------------------------------------------------------
enum Kind { K_setup_prop, K_setup_pos, K_probe_fft, K_forward, K_loss, K_finalize, K_zero, K_backward, K_gather_object,
            K_reduce_probe, K_probe_ifft, K_dohat, K_axpy, K_pos_sgd, K_lsqml_alpha, K_lsqml_object, K_lsqml_probe,
            K_lsqml_pos, K_bilinear_patches, K_pos_bilinear, K_epie_max, K_alpha_pos, K_gather_willum, K_objtrans, K_regularizer, K_constraint, K_adam, K_step_object, K_step_probe, K_single, K_COUNT };
const char* const kKindNames[K_COUNT] = {"k_setup_prop", "k_setup_pos", "k_probe_fft", "k_forward", "k_loss", "k_finalize",
                                         "k_zero", "k_backward", "k_gather_object", "k_reduce_probe", "k_probe_ifft", "k_dohat",
                                         "k_axpy", "k_pos_sgd", "k_lsqml_alpha", "k_lsqml_object", "k_lsqml_probe", "k_lsqml_pos",
                                         "k_bilinear_patches", "k_pos_bilinear", "k_epie_max", "k_alpha_pos", "k_gather_willum", "k_objtrans", "k_regularizer", "k_constraint", "k_adam", "k_step_object", "k_step_probe", "k_single"};

inline void prof_mark(int kind, cudaStream_t st) {
  if (!g_prof_on) return;
  ProfMark m; m.kind = kind;
  if (cudaEventCreate(&m.ev) != cudaSuccess) return;
  cudaEventRecord(m.ev, st);
  g_prof.push_back(m);
}

#define LAUNCH_CHECK(kind, st)                                  \
  do {                                                          \
    ++g_launches;                                               \
    if (cudaGetLastError() != cudaSuccess) return PT_ERR_CUDA;  \
    prof_mark(kind, st);                                        \
  } while (0)

int validate(const pt_problem* p) {
  if (!p) return PT_ERR_NULL;
  if (p->n != 64 && p->n != 128 && p->n != 256) return PT_ERR_BAD_SIZE;
  if (p->n_modes < 1 || p->n_slices < 1 || p->n_batch < 1 || p->n_pos_total < p->n_batch) return PT_ERR_BAD_SIZE;
  if (p->obj_ny < p->n || p->obj_nx < p->n) return PT_ERR_BAD_SIZE;
  if (!(p->pixel_size > 0.f) || !(p->wavelength > 0.f) || !(p->eps > 0.f)) return PT_ERR_BAD_PARAM;
  if (p->loss != PT_LOSS_AMPLITUDE && p->loss != PT_LOSS_POISSON && p->loss != PT_LOSS_GAUSSIAN) return PT_ERR_BAD_PARAM;
  if (p->loss == PT_LOSS_GAUSSIAN && !(p->loss_c > 0.f)) return PT_ERR_BAD_PARAM;
  if (p->shift_mode != PT_SHIFT_FOURIER_PROBE && p->shift_mode != PT_SHIFT_BILINEAR_OBJECT) return PT_ERR_BAD_PARAM;
  if (p->shift_mode == PT_SHIFT_BILINEAR_OBJECT && (p->obj_ny < p->n + 1 || p->obj_nx < p->n + 1)) return PT_ERR_BAD_SIZE;
  if (p->n_slices > 1 && !p->slice_thickness) return PT_ERR_NULL;
  if (p->loss_c < 0.f) return PT_ERR_BAD_PARAM;
  return PT_OK;
}

KP make_kp(const pt_problem* p, const Ws& w, const pt_c64* object, const pt_c64* probe, const float* positions,
           const float* intensity, const int32_t* batch_idx) {
  KP k;
  k.N = p->n; k.M = p->n_modes; k.Mg = p->n_modes; k.Mi = p->n_modes; k.S = p->n_slices; k.ony = p->obj_ny; k.onx = p->obj_nx; k.J = p->n_batch; k.Jtot = p->n_pos_total;
  k.j0 = 0; k.jc = 0; k.px = p->pixel_size;
  k.chi_scale = (p->flags & PT_LSQML_MODULUS_CHI) ? 2.0f : 1.0f;
  const double lim = 0.5 * (double)p->bandlimit * (double)p->n;
  k.bandlim2 = p->bandlimit > 0.f ? (float)(lim * lim) : -1.0f;
  k.loss = p->loss; k.loss_c = p->loss_c; k.eps = p->eps;
  k.bilinear = p->shift_mode == PT_SHIFT_BILINEAR_OBJECT;
  k.object = (const cf*)object; k.probe = (const cf*)probe; k.positions = positions; k.intensity = intensity;
  k.batch_idx = batch_idx; k.w = w;
  return k;
}

// launch on `st`; CL = 4 geometries launch clusters of four consecutive CTAs (one field per cluster)
template <class G, class... KArgs, class... Args>
cudaError_t launch_fft(void (*kern)(KArgs...), unsigned grid, size_t smem, cudaStream_t st, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid, 1, 1); cfg.blockDim = dim3(G::T, 1, 1); cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = G::CL; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  cfg.attrs = at; cfg.numAttrs = G::CL > 1 ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// SMs of the current device (asked once per process and device)
inline int sm_count() {
  static std::mutex mu;
  static int cached[32] = {0};
  int dev = 0, n = 148;
  if (cudaGetDevice(&dev) != cudaSuccess) return n;
  std::lock_guard<std::mutex> lock(mu);
  if (dev < 32 && cached[dev] > 0) return cached[dev];
  if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) n = 148;
  if (dev < 32) cached[dev] = n;
  return n;
}

// dynamic shared-memory limits of the FFT kernels: set once per process and geometry (per device: the attribute is per context)
template <class G>
int set_smem_attrs_now() {
  const int b = (int)fft_smem_bytes<G>();
  const int c = (int)chain_smem_bytes<G>();
  bool ok = true;
  auto set = [&](const void* f, int bytes) { ok = ok && cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) == cudaSuccess; };
  set((const void*)k_forward<G, 0>, c); set((const void*)k_forward<G, 1>, c); set((const void*)k_forward<G, 2>, c);
  set((const void*)k_backward<G, 0, false, false>, c); set((const void*)k_backward<G, 0, true, false>, c); set((const void*)k_backward<G, 2, false, false>, c);
  set((const void*)k_backward<G, 0, false, true>, c); set((const void*)k_backward<G, 0, true, true>, c);
  set((const void*)k_backward_pair<G, 0, false, false>, c); set((const void*)k_backward_pair<G, 0, true, false>, c); set((const void*)k_backward_pair<G, 2, false, false>, c);
  set((const void*)k_backward_pair<G, 0, false, true>, c); set((const void*)k_backward_pair<G, 0, true, true>, c);
  set((const void*)k_probe_fft<G>, b); set((const void*)k_probe_ifft<G>, b); set((const void*)k_step_probe<G>, b);
  if constexpr (G::CL == 1) set((const void*)k_single<G>, c);
  return ok ? PT_OK : PT_ERR_CUDA;
}
template <class G>
int set_smem_attrs() {
  static std::mutex mu;
  static unsigned done_mask = 0;                                   // bit d: device d configured
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return PT_ERR_CUDA;
  std::lock_guard<std::mutex> lock(mu);
  if (dev < 32 && (done_mask >> dev) & 1u) return PT_OK;
  const int rc = set_smem_attrs_now<G>();
  if (rc == PT_OK && dev < 32) done_mask |= 1u << dev;
  return rc;
}

// common prologue: tables, position split, probe spectrum
template <class G>
int prologue(const pt_problem* p, KP& kp, cudaStream_t st, float* za = nullptr, size_t na = 0, float* zb = nullptr, size_t nb = 0, float* zc = nullptr, size_t nc = 0) {
  int rc = set_smem_attrs<G>();
  if (rc != PT_OK) return rc;
  const int nprop = p->n_slices - 1;
  for (int i0 = 0; i0 < nprop; i0 += 64) {
    PropArgs a;
    a.N = p->n; a.nprop = nprop - i0 < 64 ? nprop - i0 : 64; a.px = (double)p->pixel_size; a.lambda = (double)p->wavelength;
    a.tx = (double)p->tilt_x_mrad; a.ty = (double)p->tilt_y_mrad; a.hx = kp.w.hx; a.hy = kp.w.hy; a.i0 = i0;
    for (int i = 0; i < a.nprop; ++i) a.dz[i] = p->slice_thickness[i0 + i];
    const int n = a.nprop * 2 * a.N;
    k_setup_prop<<<(n + 255) / 256, 256, 0, st>>>(a);
    LAUNCH_CHECK(K_setup_prop, st);
  }
  {
    const size_t on = (size_t)p->n_slices * p->obj_ny * p->obj_nx;
    const unsigned nb_obj = (unsigned)((on + 255) / 256), per = 256u / (unsigned)p->n, nb_pos = ((unsigned)p->n_batch + per - 1) / per;
    k_pair_object<<<nb_obj + nb_pos, 256, 0, st>>>(kp, (G::CL == 1 ? 1 : 2) * G::N2X, za, na, zb, nb, zc, nc, nb_obj);
    LAUNCH_CHECK(K_setup_pos, st);
  }
  launch_fft<G>(k_probe_fft<G>, p->n_modes * G::CL, fft_smem_bytes<G>(), st, kp.probe, kp.w.Pt, 1.0f, (const float*)nullptr, 0.0f);
  LAUNCH_CHECK(K_probe_fft, st);
  return PT_OK;
}

template <class G>
int run_forward(const pt_problem* p, KP kp, double* loss_d, float* loss_per_pos_d, float* model_intensity_d, cudaStream_t st) {
  int rc = prologue<G>(p, kp, st);
  if (rc != PT_OK) return rc;
  for (int j0 = 0; j0 < p->n_batch; j0 += kp.w.Jc) {
    kp.j0 = j0; kp.jc = p->n_batch - j0 < kp.w.Jc ? p->n_batch - j0 : kp.w.Jc;
    if (kp.bilinear) { k_bilinear_patches<<<kp.jc * p->n_slices, 256, 0, st>>>(kp, (G::CL == 1 ? 1 : 2) * G::N2X); LAUNCH_CHECK(K_bilinear_patches, st); }
    launch_fft<G>(k_forward<G, 0>, kp.jc * p->n_modes * G::CL, chain_smem_bytes<G>(), st, kp);
    LAUNCH_CHECK(K_forward, st);
    k_loss<G><<<kp.jc * G::CL, G::T, 0, st>>>(kp, model_intensity_d, 0);
    LAUNCH_CHECK(K_loss, st);
  }
  if (loss_d || loss_per_pos_d) {
    k_finalize<<<1, 1024, 0, st>>>(kp, G::CL, loss_d, (p->flags & PT_ACCUMULATE) != 0, loss_per_pos_d, nullptr, nullptr);
    LAUNCH_CHECK(K_finalize, st);
  }
  return PT_OK;
}

template <class G>
int run_gradient(const pt_problem* p, KP kp, pt_c64* gO, pt_c64* gP, float* gX, float* illum, const float* illum_prev,
                 float* step_terms, double* loss_d, float* loss_per_pos_d, cudaStream_t st, const cudaEvent_t* chunk_ready) {
  // chunk_ready (ptycho_gradient_host only): one event per chunk, recorded on its copy stream when that chunk's measured
  // patterns have arrived on the device; the pass waits for chunk c's event before the first kernel that reads them (k_loss)
  const size_t NN = (size_t)p->n * p->n, on = (size_t)p->n_slices * p->obj_ny * p->obj_nx;
  const bool acc = (p->flags & PT_ACCUMULATE) != 0;
  const bool want_illum = (p->flags & PT_WANT_ILLUM) && illum;
  // tables, position split, probe spectrum; the object pre-pass also clears the probe-gradient accumulator and (unless accumulating)
  // grad_object and the illumination map(s)
  int rc = prologue<G>(p, kp, st, (float*)kp.w.gPt_acc, (size_t)p->n_modes * NN * 4, (float*)gO, acc ? 0 : on * 2, illum,
                       !acc && want_illum ? ((p->flags & PT_WANT_WEIGHTED_ILLUM) ? 2 * on : on) : 0);
  if (rc != PT_OK) return rc;
  const bool want_pos = (p->flags & PT_WANT_POS_GRAD) && gX && !(p->flags & PT_EPIE);
  const bool want_steps = (p->flags & PT_WANT_STEP_SIZES) && step_terms;
  const bool want_w = (p->flags & PT_WANT_WEIGHTED_ILLUM) != 0;     // validated by the caller: needs want_illum && want_steps
  const bool bilin = p->shift_mode == PT_SHIFT_BILINEAR_OBJECT;
  const bool epie = (p->flags & PT_EPIE) != 0;
  // two modes per CTA (cluster), their patch gradients summed on chip (k_backward_pair): needs an even number of modes
  const bool paired = use_pairs(p);
  const bool stage_il = kp.w.ilpart != nullptr && !epie;            // |Psi|^2 staged by the backward kernel (step sizes; illumination map)
  const bool h16 = (p->flags & PT_STASH_FP16) != 0;                 // validated by the caller: no ePIE, illumination map only through ilpart
  // single slice, plain gradient: forward, loss and adjoint of a position fused in one persistent kernel (k_single)
  const bool single = G::CL == 1 && p->n_slices == 1 && !bilin && !epie && !want_steps && !want_illum && !h16 && !kp.w.ilpart &&
                      !(p->flags & PT_NO_SINGLE_SLICE_FUSION);
  kp.Mg = single ? 1 : paired ? p->n_modes / 2 : p->n_modes;
  kp.Mi = paired ? p->n_modes / 2 : p->n_modes;
  const dim3 ggrid((p->obj_nx + GATHER_TW - 1) / GATHER_TW, (p->obj_ny + 256 / GATHER_TW - 1) / (256 / GATHER_TW), p->n_slices), gblock(GATHER_TW, 256 / GATHER_TW);
  // forward chain, loss, backward chain of the current chunk (kp.j0, kp.jc); the backward kernels stage gT, conj(R) G~, |Psi|^2
  int single_ctas = 0;                                              // k_single: its CTAs each leave ONE probe-partial plane per mode
  auto chains = [&](bool wait_patterns) -> int {
    if constexpr (G::CL == 1) {
      if (single) {
        if (wait_patterns && chunk_ready && cudaStreamWaitEvent(st, chunk_ready[kp.j0 / kp.w.Jc], 0) != cudaSuccess) return PT_ERR_CUDA;
        const int resident = sm_count() * min_blocks<G>();
        single_ctas = kp.jc < resident ? kp.jc : resident;
        launch_fft<G>(k_single<G>, single_ctas, chain_smem_bytes<G>(), st, kp, want_pos ? 1 : 0);
        LAUNCH_CHECK(K_single, st);
        return PT_OK;
      }
    }
    if (bilin) { k_bilinear_patches<<<kp.jc * p->n_slices, 256, 0, st>>>(kp, (G::CL == 1 ? 1 : 2) * G::N2X); LAUNCH_CHECK(K_bilinear_patches, st); }
    if (h16) launch_fft<G>(k_forward<G, 2>, kp.jc * p->n_modes * G::CL, chain_smem_bytes<G>(), st, kp);
    else launch_fft<G>(k_forward<G, 1>, kp.jc * p->n_modes * G::CL, chain_smem_bytes<G>(), st, kp);
    LAUNCH_CHECK(K_forward, st);
    if (wait_patterns && chunk_ready && cudaStreamWaitEvent(st, chunk_ready[kp.j0 / kp.w.Jc], 0) != cudaSuccess) return PT_ERR_CUDA;
    k_loss<G><<<kp.jc * G::CL, G::T, 0, st>>>(kp, nullptr, 1);
    LAUNCH_CHECK(K_loss, st);
    const int wp = want_pos && !bilin ? 1 : 0;
    if (epie) {
      k_patch_max<<<kp.jc * p->n_slices, 256, 0, st>>>(kp);
      LAUNCH_CHECK(K_epie_max, st);
      k_stash_max<<<kp.jc * p->n_modes * p->n_slices * G::CL, 256, 0, st>>>(kp.w.stash, kp.w.psimax, FL<G>::NNS);
      LAUNCH_CHECK(K_epie_max, st);
      if (paired) launch_fft<G>(k_backward_pair<G, 2, false, false>, kp.jc * (p->n_modes / 2) * G::CL, chain_smem_bytes<G>(), st, kp, 0);
      else launch_fft<G>(k_backward<G, 2, false, false>, kp.jc * p->n_modes * G::CL, chain_smem_bytes<G>(), st, kp, 0);
    } else if (paired) {
      const unsigned grid = kp.jc * (p->n_modes / 2) * G::CL;
      if (stage_il && h16) launch_fft<G>(k_backward_pair<G, 0, true, true>, grid, chain_smem_bytes<G>(), st, kp, wp);
      else if (stage_il) launch_fft<G>(k_backward_pair<G, 0, true, false>, grid, chain_smem_bytes<G>(), st, kp, wp);
      else if (h16) launch_fft<G>(k_backward_pair<G, 0, false, true>, grid, chain_smem_bytes<G>(), st, kp, wp);
      else launch_fft<G>(k_backward_pair<G, 0, false, false>, grid, chain_smem_bytes<G>(), st, kp, wp);
    } else {
      const unsigned grid = kp.jc * p->n_modes * G::CL;
      if (stage_il && h16) launch_fft<G>(k_backward<G, 0, true, true>, grid, chain_smem_bytes<G>(), st, kp, wp);
      else if (stage_il) launch_fft<G>(k_backward<G, 0, true, false>, grid, chain_smem_bytes<G>(), st, kp, wp);
      else if (h16) launch_fft<G>(k_backward<G, 0, false, true>, grid, chain_smem_bytes<G>(), st, kp, wp);
      else launch_fft<G>(k_backward<G, 0, false, false>, grid, chain_smem_bytes<G>(), st, kp, wp);
    }
    LAUNCH_CHECK(K_backward, st);
    return PT_OK;
  };
  // staged arrays that hold the whole batch: the kernels get them advanced to the chunk's first position
  const Ws w0 = kp.w;
  auto stage_chunk = [&](int j0) {
    const size_t js = w0.stage_all ? (size_t)j0 : 0, FN = (size_t)G::CL * FL<G>::NNS;
    kp.w.gTpart = w0.gTpart + js * kp.Mg * p->n_slices * FN;
    kp.w.Gpart = w0.Gpart + js * p->n_modes * FN;
    kp.w.ilpart = w0.ilpart ? w0.ilpart + js * kp.Mi * p->n_slices * FN : nullptr;
  };
  for (int j0 = 0; j0 < p->n_batch; j0 += kp.w.Jc) {
    kp.j0 = j0; kp.jc = p->n_batch - j0 < kp.w.Jc ? p->n_batch - j0 : kp.w.Jc;
    stage_chunk(j0);
    if ((rc = chains(true)) != PT_OK) return rc;
    // few tiles (small objects, single slice: configs 1 and 2): the tile gather is bound by the latency of each pixel's serial
    // walk over its windows, so the windows are split over the warps of a block instead (k_gather_object_w: config 1 0.108 -> 0.023 ms,
    // config 2 0.66 -> 0.13 ms); many tiles (configs 3-5): the tile gather is DRAM-bound and the wider tiles over-fetch less
    // (config 3: 9.6 ms against 16.9 ms).  The choice depends on the problem's dimensions only, never on the chunking.
    const dim3 wgrid((p->obj_nx + 31) / 32, p->obj_ny, p->n_slices);
    if ((size_t)ggrid.x * ggrid.y * ggrid.z < 2368) {
    if (bilin) {
      if (want_illum) k_gather_object_w<G, true, true><<<wgrid, 256, 0, st>>>(kp, (cf*)gO, illum);
      else k_gather_object_w<G, false, true><<<wgrid, 256, 0, st>>>(kp, (cf*)gO, nullptr);
    } else {
      if (want_illum) k_gather_object_w<G, true, false><<<wgrid, 256, 0, st>>>(kp, (cf*)gO, illum);
      else k_gather_object_w<G, false, false><<<wgrid, 256, 0, st>>>(kp, (cf*)gO, nullptr);
    }
    } else
    if (bilin) {
      if (want_illum) k_gather_object<G, true, true><<<ggrid, gblock, 0, st>>>(kp, (cf*)gO, illum);
      else k_gather_object<G, false, true><<<ggrid, gblock, 0, st>>>(kp, (cf*)gO, nullptr);
    } else {
      if (want_illum) k_gather_object<G, true, false><<<ggrid, gblock, 0, st>>>(kp, (cf*)gO, illum);
      else k_gather_object<G, false, false><<<ggrid, gblock, 0, st>>>(kp, (cf*)gO, nullptr);
    }
    LAUNCH_CHECK(K_gather_object, st);
    if (bilin && want_pos) {
      k_pos_bilinear<G><<<kp.jc, 256, 0, st>>>(kp, G::CL);
      LAUNCH_CHECK(K_pos_bilinear, st);
    }
    KP kr = kp;
    if (single) kr.jc = single_ctas;                                 // the planes of the fused single-slice kernel are per CTA, not per position
    k_reduce_probe<<<dim3((unsigned)((NN + 255) / 256), p->n_modes, kReduceZ), 256, 0, st>>>(kr, kp.w.gPt_part);
    LAUNCH_CHECK(K_reduce_probe, st);
    k_reduce_probe2<<<dim3((unsigned)((NN + 255) / 256), p->n_modes), 256, 0, st>>>(kp, kp.w.gPt_part);
    LAUNCH_CHECK(K_reduce_probe, st);
  }
  launch_fft<G>(k_probe_ifft<G>, p->n_modes * G::CL, fft_smem_bytes<G>(), st, (const double2*)kp.w.gPt_acc, (cf*)gP, acc ? 1 : 0,
                epie ? 1.0 / (double)p->n_batch : 1.0);                         // ePIE: probe direction averaged over the group
  LAUNCH_CHECK(K_probe_ifft, st);
  if (want_steps) {
    // H14 (O13/O14): needs the batch-aggregated gO, gP, and what the backward pass staged for every position of the batch
    k_dohat<<<(unsigned)((on + 255) / 256), 256, 0, st>>>((const cf*)gO, illum_prev, p->lsqml_delta_o, kp.w.dOhat, on);
    LAUNCH_CHECK(K_dohat, st);
    launch_fft<G>(k_probe_fft<G>, p->n_modes * G::CL, fft_smem_bytes<G>(), st, (const cf*)gP, kp.w.Qt, -1.0f / (p->lsqml_delta_p + 1.0f),
               p->lsqml_probe_precond_d, p->lsqml_delta_p);
    LAUNCH_CHECK(K_probe_fft, st);
    const bool recompute = kp.w.Jc < p->n_batch && !kp.w.stage_all;      // the staged arrays hold the last chunk only
    for (int j0 = 0; j0 < p->n_batch; j0 += kp.w.Jc) {
      kp.j0 = j0; kp.jc = p->n_batch - j0 < kp.w.Jc ? p->n_batch - j0 : kp.w.Jc;
      stage_chunk(j0);
      if (recompute) { if ((rc = chains(false)) != PT_OK) return rc; }
      else if (bilin && kp.w.Jc < p->n_batch) { k_bilinear_patches<<<kp.jc * p->n_slices, 256, 0, st>>>(kp, (G::CL == 1 ? 1 : 2) * G::N2X); LAUNCH_CHECK(K_bilinear_patches, st); }
      if (bilin) k_step_object<G, true><<<kp.jc * p->n_slices, 256, 0, st>>>(kp);
      else k_step_object<G, false><<<kp.jc * p->n_slices, 256, 0, st>>>(kp);
      LAUNCH_CHECK(K_step_object, st);
      launch_fft<G>(k_step_probe<G>, kp.jc * p->n_modes * G::CL, fft_smem_bytes<G>(), st, kp);
      LAUNCH_CHECK(K_step_probe, st);
      if (want_w) {   // PAPER.md:225 with per-position step sizes (R24): W += sum_j alpha_{O,i,j} sum_k |Psi_{i,k,j}|^2
        k_alpha_pos<<<(kp.jc * p->n_slices + 255) / 256, 256, 0, st>>>(kp, p->lsqml_gamma);
        LAUNCH_CHECK(K_alpha_pos, st);
        k_gather_willum<G><<<ggrid, gblock, 0, st>>>(kp, illum + on);
        LAUNCH_CHECK(K_gather_willum, st);
      }
    }
  }
  k_finalize<<<1, 1024, 0, st>>>(kp, G::CL, loss_d, acc ? 1 : 0, loss_per_pos_d, want_pos ? gX : nullptr, want_steps ? step_terms : nullptr);
  LAUNCH_CHECK(K_finalize, st);
  return PT_OK;
}

// rows compacted on the device (ptycho_gradient_host with an index list): out[j] = table[rows[j]]
__global__ void k_gather_rows(const float2* table, const int32_t* rows, float2* out, int J) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j < J) out[j] = table[rows[j]];
}

// ptycho_gradient_host's copy stream and events: created once per device, reused by later calls, never destroyed (the only
// process-wide state of the library; the lock serialises concurrent host-path calls)
struct HostPoolDev { int dev; cudaStream_t copy; cudaEvent_t start; std::vector<cudaEvent_t> ready; };
struct HostPool {
  std::mutex mu;
  std::vector<HostPoolDev> devs;
  HostPoolDev* cur = nullptr;
  bool acquire(size_t nchunk) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return false;
    cur = nullptr;
    for (auto& d : devs) if (d.dev == dev) cur = &d;
    if (!cur) {
      HostPoolDev d; d.dev = dev; d.copy = nullptr; d.start = nullptr;
      if (cudaStreamCreateWithFlags(&d.copy, cudaStreamNonBlocking) != cudaSuccess) return false;
      if (cudaEventCreateWithFlags(&d.start, cudaEventDisableTiming) != cudaSuccess) return false;
      devs.push_back(d);
      cur = &devs.back();
    }
    while (cur->ready.size() < nchunk) {
      cudaEvent_t e;
      if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) return false;
      cur->ready.push_back(e);
    }
    return true;
  }
};
HostPool& host_pool() { static HostPool hp; return hp; }

int32_t gradient_impl(const pt_problem* p, const pt_c64* object_d, const pt_c64* probe_d, const float* positions_d,
                        const float* intensity_d, const int32_t* batch_idx_d, pt_c64* grad_object_d, pt_c64* grad_probe_d,
                        float* grad_pos_d, float* illum_d, const float* illum_prev_d, float* step_terms_d, double* loss_d,
                        float* loss_per_pos_d, void* workspace_d, size_t workspace_bytes, void* cuda_stream, const cudaEvent_t* chunk_ready) {
  int rc = validate(p);
  if (rc != PT_OK) return rc;
  if (!object_d || !probe_d || !positions_d || !intensity_d || !grad_object_d || !grad_probe_d || !workspace_d) return PT_ERR_NULL;
  if ((p->flags & PT_WANT_STEP_SIZES) && step_terms_d && !illum_prev_d) return PT_ERR_NULL;
  // PT_LSQML_MODULUS_CHI: the wavefront update of PAPER.md:173 is given for the amplitude model only
  if ((p->flags & PT_LSQML_MODULUS_CHI) && p->loss != PT_LOSS_AMPLITUDE) return PT_ERR_UNSUPPORTED;
  if (p->flags & PT_WANT_WEIGHTED_ILLUM) {
    if (!(p->flags & PT_WANT_ILLUM) || !(p->flags & PT_WANT_STEP_SIZES) || (p->flags & PT_EPIE)) return PT_ERR_BAD_PARAM;
    if (p->shift_mode == PT_SHIFT_BILINEAR_OBJECT) return PT_ERR_UNSUPPORTED;   // the weighted map is gathered over integer windows
    if (!illum_d || !step_terms_d) return PT_ERR_NULL;
    if (!(p->lsqml_gamma >= 0.f)) return PT_ERR_BAD_PARAM;
  }
  // ePIE directions (the optimal wavefront update is given for the amplitude model): amplitude loss,
  // Fourier-shift mode, no step-size terms, no position gradient
  if ((p->flags & PT_EPIE) && (p->loss != PT_LOSS_AMPLITUDE || p->shift_mode != PT_SHIFT_FOURIER_PROBE ||
                               ((p->flags & PT_WANT_STEP_SIZES) && step_terms_d) || ((p->flags & PT_WANT_POS_GRAD) && grad_pos_d)))
    return PT_ERR_UNSUPPORTED;
  Ws w;
  pt_problem q = *p;
  if (!step_terms_d) q.flags &= ~PT_WANT_STEP_SIZES;
  rc = ws_layout(&q, workspace_d, workspace_bytes, &w);
  if (rc != PT_OK) return rc;
  // PT_STASH_FP16: only the chain kernels read the reduced-precision stash; the two other readers (ePIE maxima, the illumination
  // map when |Psi|^2 is not staged by the backward kernel) are refused
  if ((p->flags & PT_STASH_FP16) && ((p->flags & PT_EPIE) || ((p->flags & PT_WANT_ILLUM) && illum_d && !w.ilpart))) return PT_ERR_UNSUPPORTED;
  KP kp = make_kp(&q, w, object_d, probe_d, positions_d, intensity_d, batch_idx_d);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  prof_mark(-1, st);
  const GradArgs ga = {grad_object_d, grad_probe_d, grad_pos_d, illum_d, illum_prev_d, step_terms_d, loss_d, loss_per_pos_d, chunk_ready};
  return p->n == 128 ? ptk_geo::run_gradient_128(&q, &kp, &ga, st) : p->n == 64 ? ptk_geo::run_gradient_64(&q, &kp, &ga, st)
                                                                                 : ptk_geo::run_gradient_256(&q, &kp, &ga, st);
}

}  // namespace

#define PTK_DEFINE_GEO(n)                                                                                                          \
  int ptk_geo::run_forward_##n(const pt_problem* p, const void* kp, double* loss_d, float* loss_per_pos_d, float* model_intensity_d, \
                               cudaStream_t st) {                                                                                  \
    return run_forward<Geo<n>>(p, *(const KP*)kp, loss_d, loss_per_pos_d, model_intensity_d, st);                                   \
  }                                                                                                                                \
  int ptk_geo::run_gradient_##n(const pt_problem* p, const void* kp, const GradArgs* a, cudaStream_t st) {                          \
    return run_gradient<Geo<n>>(p, *(const KP*)kp, a->gO, a->gP, a->gX, a->illum, a->illum_prev, a->step_terms, a->loss,            \
                                a->loss_per_pos, st, a->chunk_ready);                                                               \
  }
#if PTK_HAS_GEO(64)
PTK_DEFINE_GEO(64)
#endif
#if PTK_HAS_GEO(128)
PTK_DEFINE_GEO(128)
#endif
#if PTK_HAS_GEO(256)
PTK_DEFINE_GEO(256)
#endif

#if PTK_HAS_ABI
// ==================================================================================================
// C ABI
// ==================================================================================================
extern "C" {

size_t ptycho_workspace_min_bytes(const pt_problem* p) {
  if (validate(p) != PT_OK) return 0;
  const WsSizes z = ws_sizes(p);
  return z.fixed + z.per_chunk + z.per_staged + (z.il_needed ? z.per_il : 0);
}

int32_t ptycho_positions_in_flight(const pt_problem* p, size_t workspace_bytes) {
  if (validate(p) != PT_OK) return 0;
  return (int32_t)plan_chunks(p, workspace_bytes).jc;
}

size_t ptycho_workspace_bytes(const pt_problem* p) {
  if (validate(p) != PT_OK) return 0;
  const WsSizes z = ws_sizes(p);
  const size_t pp = z.per_chunk + z.per_staged + z.per_il;   // the recommendation includes the optional staging of the illumination map
  const size_t cap = (size_t)49 << 30;   // config 3: 1554 positions = 84 / 42 whole waves of forward / paired-backward CTAs
  const size_t J = p->n_batch;
  if (z.fixed + J * pp <= cap) return z.fixed + J * pp;
  // whole waves of 148 CTAs per chunk where possible (the paired backward kernel launches half as many CTAs: keep that count a
  // whole number of waves too)
  auto whole_waves = [&](size_t jc) {
    const size_t wave = 148, per_pos_ctas = staged_planes(p) * cluster_of(p->n);
    size_t pairs = jc * per_pos_ctas;
    if (pairs > wave) { pairs -= pairs % wave; jc = pairs / per_pos_ctas; }
    return jc < 1 ? (size_t)1 : jc;
  };
  if (z.il_needed) {
    // step sizes: what the backward pass stages is kept for the WHOLE batch (the sweep then needs no second pass through the
    // chain) as long as the total stays below 150 GiB; the positions in flight get the usual 49 GiB on top
    const size_t staged = J * (z.per_staged + z.per_il), big = (size_t)150 << 30;
    if (z.fixed + staged < big) {
      size_t jc = whole_waves(cap / pp);
      if (jc > J) jc = J;
      size_t room = big - z.fixed - staged;
      if (jc * z.per_chunk > room) jc = room / z.per_chunk;
      if (jc >= (J < 64 ? J : 64)) return z.fixed + staged + jc * z.per_chunk;
    }
  }
  return z.fixed + whole_waves((cap - z.fixed) / pp) * pp;
}

int32_t ptycho_forward_loss(const pt_problem* p, const pt_c64* object_d, const pt_c64* probe_d, const float* positions_d,
                            const float* intensity_d, const int32_t* batch_idx_d, double* loss_d, float* loss_per_pos_d,
                            float* model_intensity_d, void* workspace_d, size_t workspace_bytes, void* cuda_stream) {
  int rc = validate(p);
  if (rc != PT_OK) return rc;
  if (!object_d || !probe_d || !positions_d || !workspace_d) return PT_ERR_NULL;
  Ws w;
  pt_problem q = *p; q.flags &= ~PT_WANT_STEP_SIZES;
  rc = ws_layout(&q, workspace_d, workspace_bytes, &w);
  if (rc != PT_OK) return rc;
  KP kp = make_kp(p, w, object_d, probe_d, positions_d, intensity_d, batch_idx_d);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  prof_mark(-1, st);
  return p->n == 128 ? ptk_geo::run_forward_128(p, &kp, loss_d, loss_per_pos_d, model_intensity_d, st)
       : p->n == 64 ? ptk_geo::run_forward_64(p, &kp, loss_d, loss_per_pos_d, model_intensity_d, st)
                    : ptk_geo::run_forward_256(p, &kp, loss_d, loss_per_pos_d, model_intensity_d, st);
}

int32_t ptycho_gradient(const pt_problem* p, const pt_c64* object_d, const pt_c64* probe_d, const float* positions_d,
                        const float* intensity_d, const int32_t* batch_idx_d, pt_c64* grad_object_d, pt_c64* grad_probe_d,
                        float* grad_pos_d, float* illum_d, const float* illum_prev_d, float* step_terms_d, double* loss_d,
                        float* loss_per_pos_d, void* workspace_d, size_t workspace_bytes, void* cuda_stream) {
  return gradient_impl(p, object_d, probe_d, positions_d, intensity_d, batch_idx_d, grad_object_d, grad_probe_d, grad_pos_d, illum_d,
                       illum_prev_d, step_terms_d, loss_d, loss_per_pos_d, workspace_d, workspace_bytes, cuda_stream, nullptr);
}

int32_t ptycho_apply_update(const pt_problem* p, pt_c64* object_d, pt_c64* probe_d, float* positions_d,
                            const pt_c64* grad_object_d, const pt_c64* grad_probe_d, const float* grad_pos_d,
                            const float* illum_prev_d, const float* step_terms_d, const int32_t* batch_idx_d,
                            const pt_update* u, void* workspace_d, size_t workspace_bytes, void* cuda_stream) {
  int rc = validate(p);
  if (rc != PT_OK) return rc;
  if (!u) return PT_ERR_NULL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  prof_mark(-1, st);
  const size_t NN = (size_t)p->n * p->n, os = (size_t)p->obj_ny * p->obj_nx, on = os * p->n_slices, pn = NN * p->n_modes;
  if (u->mode == PT_UPDATE_SGD) {
    const bool uo = object_d && grad_object_d, up = probe_d && grad_probe_d, ux = positions_d && grad_pos_d;
    const unsigned bo = uo ? (unsigned)((2 * on + 255) / 256) : 0, bp = up ? (unsigned)((2 * pn + 255) / 256) : 0, bx = ux ? (unsigned)((p->n_batch + 255) / 256) : 0;
    if (bo + bp + bx) {
      k_sgd<<<bo + bp + bx, 256, 0, st>>>((float*)object_d, (const float*)grad_object_d, -u->lr_obj, uo ? 2 * on : 0, bo, (float*)probe_d,
                                          (const float*)grad_probe_d, -u->lr_probe, up ? 2 * pn : 0, bp, positions_d, grad_pos_d, batch_idx_d,
                                          u->lr_pos, ux ? p->n_batch : 0, p->n_pos_total);
      LAUNCH_CHECK(K_axpy, st);
    }
    return PT_OK;
  }
  if (u->mode == PT_UPDATE_EPIE) {      // O_i += beta_object dO_i ; P_k += beta_probe dP_k
    if (object_d && grad_object_d) { k_axpy<<<(unsigned)((2 * on + 255) / 256), 256, 0, st>>>((float*)object_d, (const float*)grad_object_d, u->beta_obj, 2 * on); LAUNCH_CHECK(K_axpy, st); }
    if (probe_d && grad_probe_d) { k_axpy<<<(unsigned)((2 * pn + 255) / 256), 256, 0, st>>>((float*)probe_d, (const float*)grad_probe_d, u->beta_probe, 2 * pn); LAUNCH_CHECK(K_axpy, st); }
    return PT_OK;
  }
  if (u->mode != PT_UPDATE_LSQML && u->mode != PT_UPDATE_LSQML_WEIGHTED) return PT_ERR_BAD_PARAM;
  if (!step_terms_d || !workspace_d) return PT_ERR_NULL;
  if (workspace_bytes < 256 + (size_t)(p->n_slices + 1) * sizeof(float)) return PT_ERR_WORKSPACE;
  float* alpha = (float*)((char*)workspace_d + 256);
  // under PT_LSQML_MODULUS_CHI (R31) the update directions dOhat, dPhat carry the factor 2 of chi = -2 gPhi
  const float cs = (p->flags & PT_LSQML_MODULUS_CHI) ? 2.0f : 1.0f;
  if ((p->flags & PT_LSQML_MODULUS_CHI) && p->loss != PT_LOSS_AMPLITUDE) return PT_ERR_UNSUPPORTED;
  k_lsqml_alpha<<<p->n_slices + 1, 256, 0, st>>>(step_terms_d, p->n_batch, p->n_slices, u->gamma, alpha);
  LAUNCH_CHECK(K_lsqml_alpha, st);
  if (object_d && grad_object_d) {
    if (!illum_prev_d) return PT_ERR_NULL;
    if (u->mode == PT_UPDATE_LSQML_WEIGHTED) {
      if (!u->illum_batch_d) return PT_ERR_NULL;
      k_lsqml_object_weighted<<<(unsigned)((on + 255) / 256), 256, 0, st>>>((cf*)object_d, (const cf*)grad_object_d, illum_prev_d, u->illum_batch_d,
                                                                           u->illum_batch_d + on, cs * u->beta_obj, p->lsqml_delta_o, on);
    } else
    k_lsqml_object<<<(unsigned)((on + 255) / 256), 256, 0, st>>>((cf*)object_d, (const cf*)grad_object_d, illum_prev_d, alpha, cs * u->beta_obj, p->lsqml_delta_o, os, on);
    LAUNCH_CHECK(K_lsqml_object, st);
  }
  if (probe_d && grad_probe_d) {
    k_lsqml_probe<<<(unsigned)((pn + 255) / 256), 256, 0, st>>>((cf*)probe_d, (const cf*)grad_probe_d, alpha, p->n_slices, cs * u->beta_probe, p->lsqml_delta_p, p->lsqml_probe_precond_d, NN, pn);
    LAUNCH_CHECK(K_lsqml_probe, st);
  }
  if (positions_d) {
    k_lsqml_pos<<<(p->n_batch + 255) / 256, 256, 0, st>>>(positions_d, step_terms_d, batch_idx_d, p->n_batch, p->n_slices, p->pixel_size, u->gamma, p->n_pos_total);
    LAUNCH_CHECK(K_lsqml_pos, st);
  }
  return PT_OK;
}

int32_t ptycho_object_transparency(const pt_problem* p, const pt_c64* object_d, const float* positions_d, const int32_t* batch_idx_d,
                                   float* objtrans_d, void* workspace_d, size_t workspace_bytes, void* cuda_stream) {
  int rc = validate(p);
  if (rc != PT_OK) return rc;
  if (!object_d || !positions_d || !objtrans_d || !workspace_d) return PT_ERR_NULL;
  if (p->shift_mode != PT_SHIFT_FOURIER_PROBE) return PT_ERR_UNSUPPORTED;
  if (workspace_bytes < 256) return PT_ERR_WORKSPACE;
  Ws w; memset(&w, 0, sizeof(w));
  w.status = (int32_t*)workspace_d;
  KP kp = make_kp(p, w, object_d, nullptr, positions_d, nullptr, batch_idx_d);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  prof_mark(-1, st);
  k_objtrans<<<p->n * p->n / 256, 256, 0, st>>>(kp, objtrans_d, (p->flags & PT_ACCUMULATE) ? 1 : 0);
  LAUNCH_CHECK(K_objtrans, st);
  return PT_OK;
}

size_t ptycho_workspace_host_bytes(const pt_problem* p) {
  if (validate(p) != PT_OK) return 0;
  const size_t NN = (size_t)p->n * p->n, on = (size_t)p->n_slices * p->obj_ny * p->obj_nx, pn = NN * p->n_modes, J = p->n_batch;
  size_t s = align_up(on * 8) * 2 + align_up(pn * 8) * 2 + align_up(J * 8) * 2 + align_up(J * NN * 4) + align_up(J * 4) + 256;
  s += align_up((size_t)p->n_pos_total * 8) + align_up(J * 4);           // whole position table + batch rows (batch_idx_h only)
  return s + ptycho_workspace_bytes(p);
}

int32_t ptycho_gradient_host(const pt_problem* p, const pt_c64* object_h, const pt_c64* probe_h, const float* positions_h,
                             const float* intensity_h, const int32_t* batch_idx_h, pt_c64* grad_object_h, pt_c64* grad_probe_h,
                             float* grad_pos_h, double* loss_h, float* loss_per_pos_h, void* workspace_d, size_t workspace_bytes,
                             void* cuda_stream) {
  int rc = validate(p);
  if (rc != PT_OK) return rc;
  if (!object_h || !probe_h || !positions_h || !intensity_h || !grad_object_h || !grad_probe_h || !workspace_d) return PT_ERR_NULL;
  if (workspace_bytes < ptycho_workspace_host_bytes(p)) return PT_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t NN = (size_t)p->n * p->n, on = (size_t)p->n_slices * p->obj_ny * p->obj_nx, pn = NN * p->n_modes, J = p->n_batch;
  if (batch_idx_h)
    for (size_t j = 0; j < J; ++j)
      if (batch_idx_h[j] < 0 || batch_idx_h[j] >= p->n_pos_total) return PT_ERR_OUT_OF_BOUNDS;   // host index list: checked here
  char* c = (char*)workspace_d; size_t off = 0;
  auto take = [&](size_t n) { char* r = c + off; off += align_up(n); return (void*)r; };
  pt_c64* obj_d = (pt_c64*)take(on * 8); pt_c64* gO_d = (pt_c64*)take(on * 8);
  pt_c64* pr_d = (pt_c64*)take(pn * 8); pt_c64* gP_d = (pt_c64*)take(pn * 8);
  float* pos_d = (float*)take(J * 8); float* gX_d = (float*)take(J * 8);
  float* int_d = (float*)take(J * NN * 4); float* lpp_d = (float*)take(J * 4);
  double* loss_d = (double*)take(256);
  float* postab_d = (float*)take((size_t)p->n_pos_total * 8); int32_t* rows_d = (int32_t*)take(J * 4);
  void* ws = c + off;                                                    // the gradient pass's own workspace (status word first)
  pt_problem q = *p;
  q.n_pos_total = (int32_t)J; q.flags &= ~(PT_ACCUMULATE | PT_WANT_STEP_SIZES | PT_WANT_ILLUM | PT_WANT_WEIGHTED_ILLUM | PT_EPIE);
  if (grad_pos_h) q.flags |= PT_WANT_POS_GRAD;
  // The measured patterns (the bulk of the input) travel on a second stream, chunk by chunk in the order the gradient pass
  // consumes them, so that all but the first chunk's copy overlaps the chain kernels; object, probe and positions go first
  // on the caller's stream.  The batch rows are compacted on the way in: the device sees rows 0..J-1.
  const size_t Jc = (size_t)ptycho_positions_in_flight(&q, workspace_bytes - off);
  if (Jc == 0) return PT_ERR_WORKSPACE;
  const size_t nchunk = (J + Jc - 1) / Jc;
  // the copy stream and the per-chunk events are created once per device and reused (the call is synchronous: it holds the
  // pool's lock until its final stream synchronisation)
  HostPool& hp = host_pool();
  std::lock_guard<std::mutex> lock(hp.mu);
  if (!hp.acquire(nchunk)) return PT_ERR_CUDA;
  cudaStream_t cs2 = hp.cur->copy;
  cudaEvent_t* ready = hp.cur->ready.data();
  // the copy stream starts after whatever the caller's stream has queued so far (the buffers may still be in use)
  bool ok = cudaEventRecord(hp.cur->start, st) == cudaSuccess && cudaStreamWaitEvent(cs2, hp.cur->start, 0) == cudaSuccess;
  ok = ok && cudaMemsetAsync(ws, 0, 256, st) == cudaSuccess;           // deferred status word of the pass
  ok = ok && cudaMemcpyAsync(obj_d, object_h, on * 8, cudaMemcpyHostToDevice, st) == cudaSuccess;
  ok = ok && cudaMemcpyAsync(pr_d, probe_h, pn * 8, cudaMemcpyHostToDevice, st) == cudaSuccess;
  if (!batch_idx_h) ok = ok && cudaMemcpyAsync(pos_d, positions_h, J * 8, cudaMemcpyHostToDevice, st) == cudaSuccess;
  else {   // one copy of the whole table and of the index list, rows compacted on the device
    ok = ok && cudaMemcpyAsync(postab_d, positions_h, (size_t)p->n_pos_total * 8, cudaMemcpyHostToDevice, st) == cudaSuccess;
    ok = ok && cudaMemcpyAsync(rows_d, batch_idx_h, J * 4, cudaMemcpyHostToDevice, st) == cudaSuccess;
    if (ok) { k_gather_rows<<<(unsigned)((J + 255) / 256), 256, 0, st>>>((const float2*)postab_d, rows_d, (float2*)pos_d, (int)J); LAUNCH_CHECK(K_setup_pos, st); }
  }
  for (size_t ch = 0; ok && ch < nchunk; ++ch) {
    const size_t j0 = ch * Jc, j1 = j0 + Jc < J ? j0 + Jc : J;
    if (!batch_idx_h) ok = cudaMemcpyAsync(int_d + j0 * NN, intensity_h + j0 * NN, (j1 - j0) * NN * 4, cudaMemcpyHostToDevice, cs2) == cudaSuccess;
    else
      for (size_t j = j0; ok && j < j1;) {                               // one copy per run of consecutive rows
        size_t e = j + 1;
        while (e < j1 && batch_idx_h[e] == batch_idx_h[e - 1] + 1) ++e;
        ok = cudaMemcpyAsync(int_d + j * NN, intensity_h + (size_t)batch_idx_h[j] * NN, (e - j) * NN * 4, cudaMemcpyHostToDevice, cs2) == cudaSuccess;
        j = e;
      }
    ok = ok && cudaEventRecord(ready[ch], cs2) == cudaSuccess;
  }
  if (!ok) { cudaStreamSynchronize(cs2); cudaStreamSynchronize(st); return PT_ERR_CUDA; }
  rc = gradient_impl(&q, obj_d, pr_d, pos_d, int_d, nullptr, gO_d, gP_d, grad_pos_h ? gX_d : nullptr, nullptr, nullptr, nullptr,
                     loss_d, lpp_d, ws, workspace_bytes - off, st, ready);
  if (rc != PT_OK) { cudaStreamSynchronize(cs2); cudaStreamSynchronize(st); return rc; }
  int32_t status_h = 0;
  ok = cudaMemcpyAsync(grad_object_h, gO_d, on * 8, cudaMemcpyDeviceToHost, st) == cudaSuccess;
  ok = ok && cudaMemcpyAsync(grad_probe_h, gP_d, pn * 8, cudaMemcpyDeviceToHost, st) == cudaSuccess;
  if (grad_pos_h) ok = ok && cudaMemcpyAsync(grad_pos_h, gX_d, J * 8, cudaMemcpyDeviceToHost, st) == cudaSuccess;
  if (loss_h) ok = ok && cudaMemcpyAsync(loss_h, loss_d, 8, cudaMemcpyDeviceToHost, st) == cudaSuccess;
  if (loss_per_pos_h) ok = ok && cudaMemcpyAsync(loss_per_pos_h, lpp_d, J * 4, cudaMemcpyDeviceToHost, st) == cudaSuccess;
  ok = ok && cudaMemcpyAsync(&status_h, ws, 4, cudaMemcpyDeviceToHost, st) == cudaSuccess;
  const bool synced = cudaStreamSynchronize(st) == cudaSuccess;       // every copy-stream event has been waited for by now
  if (!(ok && synced)) return PT_ERR_CUDA;
  if (status_h & kStatusOOB) return PT_ERR_OUT_OF_BOUNDS;              // the window was clamped (R4): the results are not the model's
  if (status_h & kStatusNonfinite) return PT_ERR_NONFINITE;
  return PT_OK;
}

int32_t ptycho_status(void* workspace_d, void* cuda_stream) {
  if (!workspace_d) return PT_ERR_NULL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int32_t s = 0;
  if (cudaMemcpyAsync(&s, workspace_d, sizeof(s), cudaMemcpyDeviceToHost, st) != cudaSuccess) return PT_ERR_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return PT_ERR_CUDA;
  if (cudaMemsetAsync(workspace_d, 0, sizeof(s), st) != cudaSuccess) return PT_ERR_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return PT_ERR_CUDA;
  if (s & kStatusOOB) return PT_ERR_OUT_OF_BOUNDS;
  if (s & kStatusNonfinite) return PT_ERR_NONFINITE;
  return PT_OK;
}

int64_t ptycho_launch_count(void) { return g_launches; }

int32_t ptycho_profile_enable(int32_t on) {
  for (auto& m : g_prof) cudaEventDestroy(m.ev);
  g_prof.clear();
  g_prof_on = on != 0;
  return PT_OK;
}

// Measured FP32 FMA throughput (bench.py's roofline.peak_measured): register-only FFMA chains, 16 independent accumulators
// per thread, 1024 threads x 2 blocks per SM; best of five launches timed with CUDA events.
__global__ void __launch_bounds__(1024, 2) k_ffma_peak(float* out, float a, float b, int iters) {
  float x[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) x[i] = (float)(threadIdx.x + i);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int i = 0; i < 16; ++i) x[i] = fmaf(x[i], a, b);
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += x[i];
  if (s == 12345.678f) out[0] = s;                                  // never true for the a, b passed: keeps the chains alive
}
int32_t ptycho_profile_fp32_peak(double* tflops_h, void* workspace_d, void* cuda_stream) {
  if (!tflops_h || !workspace_d) return PT_ERR_NULL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return PT_ERR_CUDA;
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return PT_ERR_CUDA;
  const int iters = 8192, blocks = 2 * sms;
  double best = 0.0;
  for (int rep = 0; rep < 6; ++rep) {
    cudaEventRecord(e0, st);
    k_ffma_peak<<<blocks, 1024, 0, st>>>((float*)workspace_d + 64, 0.999f, 0.001f, iters);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); return PT_ERR_CUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double fl = 2.0 * 64.0 * iters * 1024.0 * blocks;
    if (rep > 0 && ms > 0.f && fl / (ms * 1e-3) / 1e12 > best) best = fl / (ms * 1e-3) / 1e12;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  *tflops_h = best;
  return PT_OK;
}

int32_t ptycho_profile_num_kernels(void) { return K_COUNT; }

const char* ptycho_profile_kernel_name(int32_t kind) { return kind >= 0 && kind < K_COUNT ? kKindNames[kind] : ""; }

int32_t ptycho_profile_read(float* ms_h, int64_t* launches_h) {
  if (!ms_h || !launches_h) return PT_ERR_NULL;
  for (int k = 0; k < K_COUNT; ++k) { ms_h[k] = 0.f; launches_h[k] = 0; }
  for (size_t i = 0; i < g_prof.size(); ++i) {
    if (cudaEventSynchronize(g_prof[i].ev) != cudaSuccess) return PT_ERR_CUDA;
    if (g_prof[i].kind < 0 || i == 0) continue;
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, g_prof[i - 1].ev, g_prof[i].ev) != cudaSuccess) return PT_ERR_CUDA;
    ms_h[g_prof[i].kind] += ms;
    launches_h[g_prof[i].kind] += 1;
  }
  for (auto& m : g_prof) cudaEventDestroy(m.ev);
  g_prof.clear();
  return PT_OK;
}

const char* ptycho_strerror(int32_t code) {
  switch (code) {
    case PT_OK: return "ok";
    case PT_ERR_NULL: return "null pointer";
    case PT_ERR_BAD_SIZE: return "unsupported or inconsistent size";
    case PT_ERR_BAD_PARAM: return "bad parameter";
    case PT_ERR_WORKSPACE: return "workspace too small";
    case PT_ERR_CUDA: return "CUDA error";
    case PT_ERR_OUT_OF_BOUNDS: return "a probe window leaves the object";
    case PT_ERR_NONFINITE: return "non-finite loss";
    case PT_ERR_UNSUPPORTED: return "not supported by this build";
    case PT_ERR_STATIC_LIMIT: return "the field needs more scratch than the library's static array holds (PT_STATIC_SCRATCH_BYTES): use the entry point that takes a workspace";
    default: return "unknown error";
  }
}

}  // extern "C"

#include "regularizers.cuh"
#endif  // PTK_HAS_ABI

// Geometry kernel: steps a1-a5 of DESIGN.md section 1, one thread per extrinsic sample, always fp64.
//   a1 F_k = F+ + i Fx from (ra, dec, psi), GMST and the response tensor D_k   (reading G2; F_k of Eq. (D2)-(D3),
//      PAPER.md:763-766)
//   a2 Y_lm = -2Y_lm(iota, -phi_ref) from the per-mode term tables built at create   (reading G3)
//   a3 dt_k = -(r_k . n)/c, s_k = floor(dt_k/delta_t + 1/2), pinned operation order   (reading G4; t_k of Eq. (D2))
//   a4 q = (c^2/4) sum_k [ |F_k|^2 Y^dag U_k Y + Re(F_k^2 Y^T V_k Y) ]               (Eq. (D3))
//   a5 coefficient vector B_{k,lm} = F_k Y_lm, so that Re sum conj(B) Q = sum (B.re Q.re + B.im Q.im)
#include <cuda_fp16.h>

#include "rift_internal.h"

namespace {

constexpr int GEOM_THREADS = 128;
static_assert(GEOM_THREADS * sizeof(double) == RIFT_QP_AMP_STRIDE, "amplitude column stride of the pair program");

__device__ __forceinline__ double ipow4(double p1, double p2, double p4, double p8, int e) {   // x^e, 0 <= e < 16
  double r = (e & 1) ? p1 : 1.0;
  if (e & 2) r *= p2;
  if (e & 4) r *= p4;
  if (e & 8) r *= p8;
  return r;
}

// a1-a4 for one sample.  Outputs: shifts s_k, F_k, Y_lm (arrays sized by the caller), c = D_ref/D (NaN for an invalid
// sample) and the quadratic term q.  `modes` and `Up`/`Vp` (the point's [K][M][M] blocks) may live in shared memory.
// QUAD = false leaves a4 to quad_prog (below): q_out is 0, the real amplitudes d_a of Y_a = d_a z^{m_a} go to
// amp_s[a * GEOM_THREADS] (the thread's column of a shared-memory array) and z = e^{-i phi} to z_out[0..1].
template <int MAXM, int MAXK, bool QUAD = true>
__device__ __forceinline__ void sample_geometry(const DetGeom &g, const ModeEntry *__restrict__ modes, double ra, double dec,
                                                double psi, double iota, double phi, double dist,
                                                const double2 *__restrict__ Up, const double2 *__restrict__ Vp,
                                                int32_t (&shift)[MAXK], double (&Fre)[MAXK], double (&Fim)[MAXK],
                                                double (&Yre)[MAXM], double (&Yim)[MAXM], double &c_out, double &q_out,
                                                double *amp_s = nullptr, double *z_out = nullptr) {
  const int K = g.n_det, M = g.n_modes;
  const int m_end = (MAXM <= 16) ? MAXM : M;        // unrolled (and predicated on a < M) for small MAXM, runtime bound else
  double sd, cd, sh, ch, sp, cp;
  sincos(dec, &sd, &cd);
  sincos(ra - g.gmst, &sh, &ch);           // ch = cos(ra-gmst) = cos(gha), sh = sin(ra-gmst) = -sin(gha)
  sincos(psi, &sp, &cp);

  // ---- a3: delays and integer shifts, every operation individually rounded (no FMA contraction)
  const double nx = __dmul_rn(cd, ch), ny = __dmul_rn(cd, sh), nz = sd;
#pragma unroll
  for (int k = 0; k < MAXK; ++k) {
    if (k < K) {
      const double dot = __dadd_rn(__dadd_rn(__dmul_rn(g.loc[k][0], nx), __dmul_rn(g.loc[k][1], ny)),
                                   __dmul_rn(g.loc[k][2], nz));
      const double dt = -__ddiv_rn(dot, RIFT_C_LIGHT);
      const double x = __ddiv_rn(dt, g.delta_t);
      shift[k] = (int32_t)floor(__dadd_rn(x, 0.5));
    }
  }

  // ---- a1: antenna factors
  const double sg = -sh, cg = ch;          // sin, cos of the Greenwich hour angle gmst - ra
  const double X[3] = {-cp * sg - sp * cg * sd, -cp * cg + sp * sg * sd, sp * cd};
  const double Yv[3] = {sp * sg - cp * cg * sd, sp * cg + cp * sg * sd, cp * cd};
  // symmetric 3x3 forms: XX - YY and XY + YX (6 independent entries each)
  const double pxx[6] = {X[0] * X[0] - Yv[0] * Yv[0], X[1] * X[1] - Yv[1] * Yv[1], X[2] * X[2] - Yv[2] * Yv[2],
                         X[0] * X[1] - Yv[0] * Yv[1], X[0] * X[2] - Yv[0] * Yv[2], X[1] * X[2] - Yv[1] * Yv[2]};
  const double pxy[6] = {2.0 * X[0] * Yv[0], 2.0 * X[1] * Yv[1], 2.0 * X[2] * Yv[2], X[0] * Yv[1] + X[1] * Yv[0],
                         X[0] * Yv[2] + X[2] * Yv[0], X[1] * Yv[2] + X[2] * Yv[1]};
#pragma unroll
  for (int k = 0; k < MAXK; ++k) {
    if (k < K) {
      const double *D = g.resp[k];
      // D need not be exactly symmetric in the caller's array: use D_ij + D_ji for the off-diagonal pairs
      const double d01 = D[1] + D[3], d02 = D[2] + D[6], d12 = D[5] + D[7];
      Fre[k] = D[0] * pxx[0] + D[4] * pxx[1] + D[8] * pxx[2] + d01 * pxx[3] + d02 * pxx[4] + d12 * pxx[5];
      Fim[k] = D[0] * pxy[0] + D[4] * pxy[1] + D[8] * pxy[2] + d01 * pxy[3] + d02 * pxy[4] + d12 * pxy[5];
    }
  }

  // ---- a2: harmonics.  The terms of one mode are coef[t] c^(pc0 - 2t) s^(ps0 + 2t) (c, s = cos, sin of iota/2), i.e.
  // c^pcmin s^psmin times a homogeneous polynomial in c^2, s^2 (Horner); integer powers and e^{-i |m| phi} by binary
  // powering -- no per-thread tables.
  {
    double s1, c1, s2h, c2h;
    sincos(0.5 * iota, &s1, &c1);
    const double c2 = c1 * c1, c4 = c2 * c2, c8 = c4 * c4;
    const double s2 = s1 * s1, s4 = s2 * s2, s8 = s4 * s4;
    sincos(phi, &s2h, &c2h);
    const double z1r = c2h, z1i = -s2h;                                   // z = e^{-i phi}
    if constexpr (!QUAD) z_out[0] = z1r, z_out[1] = z1i;
    const double z2r = z1r * z1r - z1i * z1i, z2i = 2.0 * z1r * z1i;
    const double z4r = z2r * z2r - z2i * z2i, z4i = 2.0 * z2r * z2i;
    const double z8r = z4r * z4r - z4i * z4i, z8i = 2.0 * z4r * z4i;
#pragma unroll(MAXM <= 16 ? MAXM : 1)
    for (int a = 0; a < m_end; ++a) {
      if (a < M) {
        const ModeEntry &e = modes[a];
        const int n = e.n_terms;
        double P = e.coef[0], spw = 1.0;
#pragma unroll
        for (int t = 1; t < RIFT_MAX_TERMS; ++t) {
          if (t < n) {
            spw *= s2;
            P = P * c2 + e.coef[t] * spw;
          }
        }
        const double amp = P * ipow4(c1, c2, c4, c8, e.pc[n - 1]) * ipow4(s1, s2, s4, s8, e.ps[0]);
        const int am = e.m < 0 ? -e.m : e.m;
        double wr = 1.0, wi = 0.0;                                          // z^|m|
        if (am & 1) wr = z1r, wi = z1i;
        if (am & 2) {
          const double t = wr * z2r - wi * z2i;
          wi = wr * z2i + wi * z2r;
          wr = t;
        }
        if (am & 4) {
          const double t = wr * z4r - wi * z4i;
          wi = wr * z4i + wi * z4r;
          wr = t;
        }
        if (am & 8) {
          const double t = wr * z8r - wi * z8i;
          wi = wr * z8i + wi * z8r;
          wr = t;
        }
        // e^{i m (-phi)} = z^m (m >= 0) or conj(z^|m|) (m < 0)
        Yre[a] = amp * wr;
        Yim[a] = (e.m < 0) ? -amp * wi : amp * wi;
        if constexpr (!QUAD) amp_s[a * GEOM_THREADS] = amp;
      }
    }
  }

  const bool bad = !(dist > 0.0) || isnan(ra) || isnan(dec) || isnan(psi) || isnan(iota) || isnan(phi);
  const double c = bad ? __longlong_as_double(0x7ff8000000000000LL) : g.d_ref / dist;
  c_out = c;
  if constexpr (!QUAD) {
    q_out = 0.0;
  } else {
  // ---- a4: quadratic term; U Hermitian, V symmetric: diagonal + 2 * strict upper triangle.  The mode-pair products
  // conj(Y_a) Y_b and Y_a Y_b do not depend on the detector and are formed once.
  double yuy[MAXK], yvr[MAXK], yvi[MAXK];
#pragma unroll
  for (int k = 0; k < MAXK; ++k) yuy[k] = yvr[k] = yvi[k] = 0.0;
#pragma unroll(MAXM <= 16 ? MAXM : 1)
  for (int a = 0; a < m_end; ++a) {
    if (a < M) {
      const double ar = Yre[a], ai = Yim[a];
#pragma unroll(MAXM <= 16 ? MAXM : 1)
      for (int bb = a; bb < m_end; ++bb) {
        if (bb < M) {
          const double br = Yre[bb], bi = Yim[bb];
          const double w = (bb == a) ? 1.0 : 2.0;
          const double cr = w * (ar * br + ai * bi), ci = w * (ar * bi - ai * br);      // conj(Y_a) Y_b
          const double pr = w * (ar * br - ai * bi), pi = w * (ar * bi + ai * br);      // Y_a Y_b
#pragma unroll
          for (int k = 0; k < MAXK; ++k) {
            if (k < K) {
              const double2 u = Up[(k * M + a) * M + bb], v = Vp[(k * M + a) * M + bb];
              yuy[k] += u.x * cr - u.y * ci;
              yvr[k] += v.x * pr - v.y * pi;
              yvi[k] += v.x * pi + v.y * pr;
            }
          }
        }
      }
    }
  }
  double q = 0.0;
#pragma unroll
  for (int k = 0; k < MAXK; ++k) {
    if (k < K) {
      const double f2 = Fre[k] * Fre[k] + Fim[k] * Fim[k];
      const double f2r = Fre[k] * Fre[k] - Fim[k] * Fim[k], f2i = 2.0 * Fre[k] * Fim[k];
      q += f2 * yuy[k] + (f2r * yvr[k] - f2i * yvi[k]);
    }
  }
  q_out = 0.25 * c * c * q;
  }
}

// ---- a4 by the pair program (QuadProg, rift_internal.h).  Shared-memory image of one intrinsic point:
// [n_entries][KT] double2 W | [M][GEOM_THREADS] double amplitudes.  The entry and bin tables are kernel parameters
// (constant bank, uniform loads): entry e is warp-uniform, so its W is a broadcast read and only the two amplitudes
// are per-thread.
struct QuadSmem {
  size_t uv, amp, total;
};
__host__ __device__ inline QuadSmem quad_smem(int n_entries, int K, int M) {
  QuadSmem L;
  L.uv = 0;
  L.amp = (size_t)n_entries * K * sizeof(double2);
  L.total = L.amp + (size_t)M * GEOM_THREADS * sizeof(double);
  return L;
}

__device__ __forceinline__ void quad_stage(const QuadProg &qp, int K, int32_t point, double2 *uv_s) {
  const double2 *src = qp.uv + (size_t)point * qp.n_entries * K;
  for (int i = threadIdx.x; i < qp.n_entries * K; i += GEOM_THREADS) uv_s[i] = src[i];
}

// q / (c^2 / 4) = sum_k |F_k|^2 Y^dag U_k Y + Re(F_k^2 Y^T V_k Y).  `uv` is the point's W block (shared or global memory),
// `amp` the thread's amplitude column (stride GEOM_THREADS), z = e^{-i phi}.
template <int KT>
__device__ __forceinline__ double quad_prog(const QuadProg &qp, const double2 *__restrict__ uv, const double *__restrict__ amp,
                                            double z1r, double z1i, const double (&Fre)[KT], const double (&Fim)[KT]) {
  double yuy[KT], yvr[KT], yvi[KT];
#pragma unroll
  for (int k = 0; k < KT; ++k) yuy[k] = yvr[k] = yvi[k] = 0.0;
  double zr = 1.0, zi = 0.0;
#pragma unroll 1
  for (int bi = 0; bi < qp.n_bins; ++bi) {
    const int kind = qp.bin_kind[bi], zstep = kind >> 1;
    if (zstep == 0) {
      zr = 1.0, zi = 0.0;
    } else if (zstep == 2) {
      zr = z1r, zi = -z1i;
    } else {
      const double si = (zstep == 1) ? z1i : -z1i;
      const double t = zr * z1r - zi * si;
      zi = zr * si + zi * z1r;
      zr = t;
    }
    double Sr[KT], Si[KT];
#pragma unroll
    for (int k = 0; k < KT; ++k) Sr[k] = Si[k] = 0.0;
    const int e1 = qp.bin_begin[bi + 1];
#pragma unroll 4
    for (int e = qp.bin_begin[bi]; e < e1; ++e) {
      const uint2 ab = qp.ent[e];
      const char *ac = reinterpret_cast<const char *>(amp);
      const double w = *reinterpret_cast<const double *>(ac + ab.x) * *reinterpret_cast<const double *>(ac + ab.y);
      const double2 *u = uv + e * KT;
#pragma unroll
      for (int k = 0; k < KT; ++k) {
        const double2 uk = u[k];
        Sr[k] = fma(w, uk.x, Sr[k]);
        Si[k] = fma(w, uk.y, Si[k]);
      }
    }
    if ((kind & 1) == 0) {
#pragma unroll
      for (int k = 0; k < KT; ++k) yuy[k] += zr * Sr[k] - zi * Si[k];
    } else {
#pragma unroll
      for (int k = 0; k < KT; ++k) {
        yvr[k] += zr * Sr[k] - zi * Si[k];
        yvi[k] += zr * Si[k] + zi * Sr[k];
      }
    }
  }
  double q = 0.0;
#pragma unroll
  for (int k = 0; k < KT; ++k) {
    const double f2 = Fre[k] * Fre[k] + Fim[k] * Fim[k];
    const double f2r = Fre[k] * Fre[k] - Fim[k] * Fim[k], f2i = 2.0 * Fre[k] * Fim[k];
    q += f2 * yuy[k] + (f2r * yvr[k] - f2i * yvi[k]);
  }
  return q;
}

// W of every (point, entry, detector) from the handle's U, V copies ([P][K][M][M] complex128)
__global__ void build_quad_uv_kernel(const __grid_constant__ QuadProg qp, const double2 *__restrict__ U, const double2 *__restrict__ V, int P, int K,
                                     int M, double2 *__restrict__ out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t total = (int64_t)P * qp.n_entries * K;
  if (i >= total) return;
  const int k = (int)(i % K);
  const int e = (int)((i / K) % qp.n_entries);
  const int64_t p = i / ((int64_t)K * qp.n_entries);
  const uint32_t w = qp.ent_full[e];
  const int a = w & 0xffu, b = (w >> 8) & 0xffu;
  const double2 *src = ((w >> 16) & 1u) ? V : U;
  double2 v = src[((p * K + k) * M + a) * M + b];
  if ((w >> 17) & 1u) v.y = -v.y;
  const double f = (a == b) ? 1.0 : 2.0;
  out[i] = make_double2(f * v.x, f * v.y);
}

// CT = coefficient type; MAXM = 8 (mode loops unrolled, Y in registers) or RIFT_MAX_MODES; MAXK = number of detectors.
// PROG (MAXM > 16 only): the quadratic term runs the pair program `qp`.
template <typename CT, int MAXM, int MAXK, bool PROG>
__global__ void __launch_bounds__(GEOM_THREADS)
geometry_kernel(DetGeom g, const ModeEntry *__restrict__ modes, Batch b, const double *__restrict__ p_ra,
                const double *__restrict__ p_dec, const double *__restrict__ p_psi, const double *__restrict__ p_iota,
                const double *__restrict__ p_phi, const double *__restrict__ p_dist, const double *__restrict__ U,
                const double *__restrict__ V, const __grid_constant__ QuadProg qp, Workspace ws,
                int32_t *__restrict__ shift_out, double *__restrict__ dbg_F, double *__restrict__ dbg_Y,
                const int32_t *__restrict__ perm, int stage_uv) {
  const int K = g.n_det, M = g.n_modes;
  // U, V of the intrinsic point of the block's first slot staged in shared memory when the launch provides room
  extern __shared__ double2 s_uv_g[];
  const int n_uv = K * M * M;
  int32_t point0 = -1;
  if (PROG) {
    const int64_t w0 = (int64_t)blockIdx.x * GEOM_THREADS;
    const int64_t src0 = perm ? (int64_t)perm[w0] : w0;
    point0 = b.ids[(b.g0 + src0) / b.n_per_seg];
    quad_stage(qp, K, point0, s_uv_g);
    __syncthreads();
  } else if (stage_uv) {
    const int64_t w0 = (int64_t)blockIdx.x * GEOM_THREADS;
    const int64_t src0 = perm ? (int64_t)perm[w0] : w0;
    point0 = b.ids[(b.g0 + src0) / b.n_per_seg];
    const double2 *u = reinterpret_cast<const double2 *>(U) + (int64_t)point0 * n_uv;
    const double2 *v = reinterpret_cast<const double2 *>(V) + (int64_t)point0 * n_uv;
    for (int i = threadIdx.x; i < n_uv; i += GEOM_THREADS) {
      s_uv_g[i] = u[i];
      s_uv_g[n_uv + i] = v[i];
    }
    __syncthreads();
  }
  const int64_t w = (int64_t)blockIdx.x * GEOM_THREADS + threadIdx.x;     // workspace slot (sorted position)
  if (w >= b.n) return;
  const int64_t src = perm ? (int64_t)perm[w] : w;                         // chunk-local index of the sample
  if (ws.orig) ws.orig[w] = (int32_t)src;
  if (src < 0) {                                                           // padding slot of a sorted layout: a null sample
    ws.scale_c[w] = 1.0;
    ws.quad[w] = 0.0;
    for (int k = 0; k < K; ++k) ws.shift[w * K + k] = INT32_MAX;           // excluded from the batch's shift bounds
    CT *out = reinterpret_cast<CT *>(reinterpret_cast<decltype(CT::x) *>(ws.coef) + w * ws.coef_stride);
    CT z;
    z.x = 0;
    z.y = 0;
    for (int i = 0; i < K * M; ++i) out[i] = z;
    return;
  }
  const int64_t gi = b.g0 + src;                                           // caller's sample index
  const int32_t point = b.ids[gi / b.n_per_seg];

  int32_t shift[MAXK];
  double Fre[MAXK], Fim[MAXK], Yre[MAXM], Yim[MAXM], c, q;
  const double2 *Up = reinterpret_cast<const double2 *>(U) + (int64_t)point * n_uv;
  const double2 *Vp = reinterpret_cast<const double2 *>(V) + (int64_t)point * n_uv;
  if (stage_uv && point == point0) {
    Up = s_uv_g;
    Vp = s_uv_g + n_uv;
  }
  if constexpr (PROG) {
    double *amp = reinterpret_cast<double *>(reinterpret_cast<unsigned char *>(s_uv_g) + quad_smem(qp.n_entries, K, M).amp) +
                  threadIdx.x;
    double z[2];
    sample_geometry<MAXM, MAXK, false>(g, modes, p_ra[gi], p_dec[gi], p_psi[gi], p_iota[gi], p_phi[gi], p_dist[gi], nullptr,
                                       nullptr, shift, Fre, Fim, Yre, Yim, c, q, amp, z);
    if (point == point0)
      q = quad_prog<MAXK>(qp, s_uv_g, amp, z[0], z[1], Fre, Fim);
    else
      q = quad_prog<MAXK>(qp, qp.uv + (size_t)point * qp.n_entries * K, amp, z[0], z[1], Fre, Fim);
    q *= 0.25 * c * c;
  } else {
    sample_geometry<MAXM, MAXK>(g, modes, p_ra[gi], p_dec[gi], p_psi[gi], p_iota[gi], p_phi[gi], p_dist[gi], Up, Vp, shift,
                                Fre, Fim, Yre, Yim, c, q);
  }
  int32_t *my_shift = ws.shift + w * K;
  for (int k = 0; k < K; ++k) {
    my_shift[k] = shift[k];
    if (shift_out) shift_out[gi * K + k] = shift[k];
    if (dbg_F) {
      dbg_F[(gi * K + k) * 2] = Fre[k];
      dbg_F[(gi * K + k) * 2 + 1] = Fim[k];
    }
  }
  if (dbg_Y)
    for (int a = 0; a < M; ++a) {
      dbg_Y[(gi * M + a) * 2] = Yre[a];
      dbg_Y[(gi * M + a) * 2 + 1] = Yim[a];
    }
  ws.scale_c[w] = c;
  ws.quad[w] = q;
  // ---- a5: coefficient vectors B = F_k Y_lm
  CT *out = reinterpret_cast<CT *>(reinterpret_cast<decltype(CT::x) *>(ws.coef) + w * ws.coef_stride);
  for (int k = 0; k < K; ++k)
    for (int a = 0; a < M; ++a) {
      CT v;
      v.x = Fre[k] * Yre[a] - Fim[k] * Yim[a];
      v.y = Fre[k] * Yim[a] + Fim[k] * Yre[a];
      out[k * M + a] = v;
    }
}

// Tensor-core variant: one thread per batch slot; writes the batch blob described at TcPlan (rift_internal.h).
// MT = number of modes, KT = number of detectors (compile time, so that the operand chunks are assembled in registers
// and nothing is predicated on k < K).  The mode tables and the U, V blocks of the block's (first) intrinsic point are
// staged in shared memory.
template <int MT, int KT>
__global__ void __launch_bounds__(GEOM_THREADS, 5)
geometry_tc_kernel(DetGeom g, const ModeEntry *__restrict__ modes, TcPlan tp, TcChunk ch, const double *__restrict__ p_ra,
                   const double *__restrict__ p_dec, const double *__restrict__ p_psi, const double *__restrict__ p_iota,
                   const double *__restrict__ p_phi, const double *__restrict__ p_dist, const double *__restrict__ U,
                   const double *__restrict__ V, int32_t *__restrict__ shift_out) {
  constexpr int K = KT;
  constexpr int KP = (6 * MT + 15) & ~15;                                   // contraction length, fp16 elements
  constexpr int NCH = KP / 8;                                               // 16-byte chunks per detector
  __shared__ ModeEntry s_modes[MT];
  __shared__ double2 s_U[KT * MT * MT], s_V[KT * MT * MT];
  const bool sorted = ch.key != nullptr;    // sorted variant: slots are the sorted slots, the sample comes through ch.perm
  const int64_t n_slots = (sorted ? (int64_t)ch.seg_begin[ch.n_lseg] : ch.n_batches) * RIFT_TC_NB;
  const int64_t w0 = (int64_t)blockIdx.x * GEOM_THREADS;                    // first slot of the block
  if (w0 >= n_slots) return;
  int64_t seg_first = (ch.gb0 + w0 / RIFT_TC_NB) / ch.nbps;                 // segment of the block's first slot
  if (sorted) {                                                             // last local segment that begins at or before the batch
    const int32_t b = (int32_t)(w0 / RIFT_TC_NB);
    int lo = 0, hi = ch.n_lseg - 1;
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if (ch.seg_begin[mid] <= b) lo = mid; else hi = mid - 1;
    }
    seg_first = ch.gb0 / ch.nbps + lo;
  }
  const int32_t point0 = ch.ids[seg_first];
  {
    const int32_t *src = reinterpret_cast<const int32_t *>(modes);
    int32_t *dst = reinterpret_cast<int32_t *>(s_modes);
    for (int i = threadIdx.x; i < (int)(MT * sizeof(ModeEntry) / 4); i += GEOM_THREADS) dst[i] = src[i];
    const double2 *u = reinterpret_cast<const double2 *>(U) + (int64_t)point0 * K * MT * MT;
    const double2 *v = reinterpret_cast<const double2 *>(V) + (int64_t)point0 * K * MT * MT;
    for (int i = threadIdx.x; i < K * MT * MT; i += GEOM_THREADS) {
      s_U[i] = u[i];
      s_V[i] = v[i];
    }
  }
  __syncthreads();
  const int64_t w = w0 + threadIdx.x;                                       // slot = local batch * 16 + n
  if (w >= n_slots) return;
  const int64_t lb = w / RIFT_TC_NB;
  const int n = (int)(w % RIFT_TC_NB);
  int64_t wn = w;                                                           // natural slot of the sample
  if (sorted) wn = ch.perm[w];
  const int64_t gb = ch.gb0 + wn / RIFT_TC_NB;
  const int64_t seg = gb / ch.nbps;
  const int64_t i = (gb % ch.nbps) * RIFT_TC_NB + (wn % RIFT_TC_NB);
  const bool valid = wn >= 0 && i < ch.n_per_seg;
  const int blob_words = sorted ? tp.blob_words_s : tp.blob_words;
  float *blob = ch.blob + lb * blob_words;
  uint4 *chunks = reinterpret_cast<uint4 *>(blob);                          // [K][NCH][16] x 8 halfs
  int32_t *dsh = reinterpret_cast<int32_t *>(blob + K * NCH * 64);          // [K][16]
  float *cl2 = blob + K * NCH * 64 + K * 16;                                // [16]
  if (!valid) {
    const uint4 z = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
    for (int k = 0; k < K; ++k) {
#pragma unroll
      for (int c = 0; c < NCH; ++c) chunks[(k * NCH + c) * 16 + n] = z;
      dsh[k * 16 + n] = 0;
    }
    cl2[n] = 0.f;
    ch.scale_c[w] = 0.0;
    ch.quad[w] = 0.0;
    return;
  }
  const int64_t gi = seg * ch.n_per_seg + i;
  const int32_t point = ch.ids[seg];
  const double2 *Up = s_U, *Vp = s_V;
  if (point != point0) {                                                    // a block that straddles two segments
    Up = reinterpret_cast<const double2 *>(U) + (int64_t)point * K * MT * MT;
    Vp = reinterpret_cast<const double2 *>(V) + (int64_t)point * K * MT * MT;
  }
  int32_t shift[KT];
  double Fre[KT], Fim[KT], Yre[MT], Yim[MT], c, q;
  sample_geometry<MT, KT>(g, s_modes, p_ra[gi], p_dec[gi], p_psi[gi], p_iota[gi], p_phi[gi], p_dist[gi], Up, Vp, shift,
                          Fre, Fim, Yre, Yim, c, q);
  ch.scale_c[w] = c;
  ch.quad[w] = q;
  // exponent scale of the fused kernel: its accumulators carry x * (Q scale of the point) * RIFT_TC_BSCALE
  cl2[n] = (float)(c * 1.4426950408889634 / ((double)ch.qscale[point] * RIFT_TC_BSCALE));
  if (sorted && n == 0) {                                                   // batch header: the common d_1 (clamped as the key)
    const int dm = tp.dmax[1], d = shift[KT > 1 ? 1 : 0] - shift[0];
    reinterpret_cast<int32_t *>(cl2 + 16)[0] = d < -dm ? -dm : (d > dm ? dm : d);
  }
#pragma unroll
  for (int k = 0; k < K; ++k) {
    if (shift_out) shift_out[gi * K + k] = shift[k];
    dsh[k * 16 + n] = (k == 0) ? tp.j0 + shift[0] : shift[k] - shift[0];
    // a5: B = F_k Y_lm, scaled, split into fp16 hi + lo; kappa = 2a (Re), 2a+1 (Im).  The contraction index runs over
    // [hi | hi | lo] facing the A operand's [Q_hi | Q_lo | Q_hi].
    uint16_t hv[KP];
#pragma unroll
    for (int a = 0; a < MT; ++a) {
      const double vr = (Fre[k] * Yre[a] - Fim[k] * Yim[a]) * RIFT_TC_BSCALE;
      const double vi = (Fre[k] * Yim[a] + Fim[k] * Yre[a]) * RIFT_TC_BSCALE;
      const __half hr = __double2half(vr), hi = __double2half(vi);
      const __half lr = __double2half(vr - (double)__half2float(hr)), li = __double2half(vi - (double)__half2float(hi));
      hv[2 * a] = hv[2 * MT + 2 * a] = __half_as_ushort(hr);
      hv[2 * a + 1] = hv[2 * MT + 2 * a + 1] = __half_as_ushort(hi);
      hv[4 * MT + 2 * a] = __half_as_ushort(lr);
      hv[4 * MT + 2 * a + 1] = __half_as_ushort(li);
    }
#pragma unroll
    for (int e = 6 * MT; e < KP; ++e) hv[e] = 0;
    uint4 *dst = chunks + (k * NCH) * 16 + n;
#pragma unroll
    for (int cc = 0; cc < NCH; ++cc) {
      uint4 v;
      v.x = (uint32_t)hv[8 * cc + 0] | ((uint32_t)hv[8 * cc + 1] << 16);
      v.y = (uint32_t)hv[8 * cc + 2] | ((uint32_t)hv[8 * cc + 3] << 16);
      v.z = (uint32_t)hv[8 * cc + 4] | ((uint32_t)hv[8 * cc + 5] << 16);
      v.w = (uint32_t)hv[8 * cc + 6] | ((uint32_t)hv[8 * cc + 7] << 16);
      dst[cc * 16] = v;
    }
  }
}

}  // namespace

namespace {
// Tensor-core variant for more than 8 modes: the modes are split into tp.n_sub subsets of tp.m_sub (one pass of lnl_tc each)
// and every batch gets one blob per subset, [sub][batch][blob_words], each with the subset's coefficient pieces in the
// UMMA layout followed by the (identical) shifts and exponent scales.  Generic in M (the harmonics live in local memory);
// MS = modes per subset (compile time, so that the operand chunks are assembled in registers).
// PROG: the quadratic term runs the pair program `qp` (its image of the block's first point in shared memory).
template <int KT, int MS, bool PROG>
__global__ void __launch_bounds__(GEOM_THREADS, PROG ? 5 : 1)
geometry_tcx_kernel(DetGeom g, const ModeEntry *__restrict__ modes, TcPlan tp, TcChunk ch, const double *__restrict__ p_ra,
                    const double *__restrict__ p_dec, const double *__restrict__ p_psi, const double *__restrict__ p_iota,
                    const double *__restrict__ p_phi, const double *__restrict__ p_dist, const double *__restrict__ U,
                    const double *__restrict__ V, const __grid_constant__ QuadProg qp, int32_t *__restrict__ shift_out,
                    int stage_uv) {
  constexpr int K = KT;
  constexpr int KP = (6 * MS + 15) & ~15, nch = KP / 8;
  const int M = g.n_modes;
  const bool sorted = ch.key != nullptr;    // sorted variant: slots are the sorted slots, the sample comes through ch.perm
  const int64_t n_slots = (sorted ? (int64_t)ch.seg_begin[ch.n_lseg] : ch.n_batches) * RIFT_TC_NB;
  // U, V of the block's (first) intrinsic point staged in shared memory when the launch provides room for them
  extern __shared__ double2 s_uv[];
  const int64_t w0 = (int64_t)blockIdx.x * GEOM_THREADS;
  if (w0 >= n_slots) return;
  int64_t seg_first = (ch.gb0 + w0 / RIFT_TC_NB) / ch.nbps;
  if (sorted) {                                                             // last local segment that begins at or before the batch
    const int32_t b = (int32_t)(w0 / RIFT_TC_NB);
    int lo = 0, hi = ch.n_lseg - 1;
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if (ch.seg_begin[mid] <= b) lo = mid; else hi = mid - 1;
    }
    seg_first = ch.gb0 / ch.nbps + lo;
  }
  const int32_t point0 = ch.ids[seg_first];
  const int n_uv = K * M * M;
  const QuadSmem QL = quad_smem(qp.n_entries, K, M);
  if (PROG) {
    quad_stage(qp, K, point0, s_uv);
    __syncthreads();
  } else if (stage_uv) {
    const double2 *u = reinterpret_cast<const double2 *>(U) + (int64_t)point0 * n_uv;
    const double2 *v = reinterpret_cast<const double2 *>(V) + (int64_t)point0 * n_uv;
    for (int i = threadIdx.x; i < n_uv; i += GEOM_THREADS) {
      s_uv[i] = u[i];
      s_uv[n_uv + i] = v[i];
    }
    __syncthreads();
  }
  const int64_t w = w0 + threadIdx.x;                                       // slot = local batch * 16 + n
  if (w >= n_slots) return;
  const int64_t lb = w / RIFT_TC_NB;
  const int n = (int)(w % RIFT_TC_NB);
  int64_t wn = w;                                                           // natural slot of the sample
  if (sorted) wn = ch.perm[w];
  const int64_t gb = ch.gb0 + wn / RIFT_TC_NB;
  const int64_t seg = gb / ch.nbps;
  const int64_t i = (gb % ch.nbps) * RIFT_TC_NB + (wn % RIFT_TC_NB);
  const bool valid = wn >= 0 && i < ch.n_per_seg;
  const int blob_words = sorted ? tp.blob_words_s : tp.blob_words;
  const size_t sub_stride = (size_t)(sorted ? ch.cap_sorted : ch.n_batches) * blob_words;   // floats between the blobs of two subsets
  float *blob0 = ch.blob + lb * blob_words;
  if (!valid) {
    for (int sub = 0; sub < tp.n_sub; ++sub) {
      float *blob = blob0 + sub * sub_stride;
      uint4 *chunks = reinterpret_cast<uint4 *>(blob);
      const uint4 z = make_uint4(0u, 0u, 0u, 0u);
      for (int k = 0; k < K; ++k) {
        for (int c = 0; c < nch; ++c) chunks[(k * nch + c) * 16 + n] = z;
        reinterpret_cast<int32_t *>(blob + K * nch * 64)[k * 16 + n] = 0;
      }
      blob[K * nch * 64 + K * 16 + n] = 0.f;
    }
    ch.scale_c[w] = 0.0;
    ch.quad[w] = 0.0;
    return;
  }
  const int64_t gi = seg * ch.n_per_seg + i;
  const int32_t point = ch.ids[seg];
  const double2 *Up = reinterpret_cast<const double2 *>(U) + (int64_t)point * n_uv;
  const double2 *Vp = reinterpret_cast<const double2 *>(V) + (int64_t)point * n_uv;
  if (stage_uv && point == point0) {
    Up = s_uv;
    Vp = s_uv + n_uv;
  }
  int32_t shift[KT];
  double Fre[KT], Fim[KT], Yre[RIFT_MAX_MODES], Yim[RIFT_MAX_MODES], c, q;
  if (PROG) {
    unsigned char *sm = reinterpret_cast<unsigned char *>(s_uv);
    double *amp = reinterpret_cast<double *>(sm + QL.amp) + threadIdx.x;
    double z[2];
    sample_geometry<RIFT_MAX_MODES, KT, false>(g, modes, p_ra[gi], p_dec[gi], p_psi[gi], p_iota[gi], p_phi[gi], p_dist[gi],
                                               nullptr, nullptr, shift, Fre, Fim, Yre, Yim, c, q, amp, z);
    if (point == point0)                                  // two call sites: shared-memory and global loads of W
      q = quad_prog<KT>(qp, s_uv, amp, z[0], z[1], Fre, Fim);
    else
      q = quad_prog<KT>(qp, qp.uv + (size_t)point * qp.n_entries * K, amp, z[0], z[1], Fre, Fim);
    q *= 0.25 * c * c;
  } else {
    sample_geometry<RIFT_MAX_MODES, KT>(g, modes, p_ra[gi], p_dec[gi], p_psi[gi], p_iota[gi], p_phi[gi], p_dist[gi], Up, Vp,
                                        shift, Fre, Fim, Yre, Yim, c, q);
  }
  ch.scale_c[w] = c;
  ch.quad[w] = q;
  const float cl2v = (float)(c * 1.4426950408889634 / ((double)ch.qscale[point] * RIFT_TC_BSCALE));
  if (shift_out)
    for (int k = 0; k < K; ++k) shift_out[gi * K + k] = shift[k];
  for (int sub = 0; sub < tp.n_sub; ++sub) {
    float *blob = blob0 + sub * sub_stride;
    int32_t *dsh = reinterpret_cast<int32_t *>(blob + K * nch * 64);
    blob[K * nch * 64 + K * 16 + n] = cl2v;
    if (sorted && n == 0) {                                                 // batch header: the common d_1 (clamped as the key)
      const int dm = tp.dmax[1], d = shift[KT > 1 ? 1 : 0] - shift[0];
      reinterpret_cast<int32_t *>(blob + K * nch * 64 + K * 16 + 16)[0] = d < -dm ? -dm : (d > dm ? dm : d);
    }
    double yr[MS], yi[MS];                                                  // the subset's harmonics, read once for all detectors
#pragma unroll
    for (int al = 0; al < MS; ++al) {
      const int a = sub * MS + al;
      yr[al] = (a < M) ? Yre[a] * RIFT_TC_BSCALE : 0.0;
      yi[al] = (a < M) ? Yim[a] * RIFT_TC_BSCALE : 0.0;
    }
    for (int k = 0; k < K; ++k) {
      dsh[k * 16 + n] = (k == 0) ? tp.j0 + shift[0] : shift[k] - shift[0];
      uint16_t hv[KP];
#pragma unroll
      for (int e = 6 * MS; e < KP; ++e) hv[e] = 0;
#pragma unroll
      for (int al = 0; al < MS; ++al) {
        const double vr = Fre[k] * yr[al] - Fim[k] * yi[al];
        const double vi = Fre[k] * yi[al] + Fim[k] * yr[al];
        const __half hr = __double2half(vr), hi = __double2half(vi);
        const __half lr = __double2half(vr - (double)__half2float(hr)), li = __double2half(vi - (double)__half2float(hi));
        hv[2 * al] = hv[2 * MS + 2 * al] = __half_as_ushort(hr);
        hv[2 * al + 1] = hv[2 * MS + 2 * al + 1] = __half_as_ushort(hi);
        hv[4 * MS + 2 * al] = __half_as_ushort(lr);
        hv[4 * MS + 2 * al + 1] = __half_as_ushort(li);
      }
      uint4 *dst = reinterpret_cast<uint4 *>(blob) + (k * nch) * 16 + n;
#pragma unroll
      for (int cc = 0; cc < nch; ++cc) {
        uint4 v;
        v.x = (uint32_t)hv[8 * cc + 0] | ((uint32_t)hv[8 * cc + 1] << 16);
        v.y = (uint32_t)hv[8 * cc + 2] | ((uint32_t)hv[8 * cc + 3] << 16);
        v.z = (uint32_t)hv[8 * cc + 4] | ((uint32_t)hv[8 * cc + 5] << 16);
        v.w = (uint32_t)hv[8 * cc + 6] | ((uint32_t)hv[8 * cc + 7] << 16);
        dst[cc * 16] = v;
      }
    }
  }
}
}  // namespace

namespace {
template <int MT>
cudaError_t launch_geometry_tc_m(const DetGeom &g, const ModeEntry *modes, const TcPlan &tp, const TcChunk &c,
                                 const double *const params[6], const double *U, const double *V, int32_t *shift_out,
                                 unsigned grid, cudaStream_t s) {
#define RIFT_GEOM_TC(KT)                                                                                                 \
  case KT:                                                                                                               \
    geometry_tc_kernel<MT, KT><<<grid, GEOM_THREADS, 0, s>>>(g, modes, tp, c, params[0], params[1], params[2], params[3], \
                                                              params[4], params[5], U, V, shift_out);                    \
    break;
  switch (tp.K) {
    RIFT_GEOM_TC(1) RIFT_GEOM_TC(2) RIFT_GEOM_TC(3) RIFT_GEOM_TC(4) RIFT_GEOM_TC(5)
    default: return cudaErrorInvalidValue;
  }
#undef RIFT_GEOM_TC
  return cudaGetLastError();
}
}  // namespace

namespace {
// Sorted tensor-core variant, pass 1: the shift bucket of every natural slot.  The delays are computed with exactly the
// operations of sample_geometry (a3), so that the bucket's d_1 is the d_1 the geometry kernel will find.
constexpr int KEY_THREADS = 1024;
// The bucket counts are formed per block in shared memory (a block touches at most two segments when the sorted variant is
// used) and added to the global counts with one atomic per non-empty (block, bucket): contended global atomics on a few
// thousand addresses serialise (measured: 1.6e6 of them on 5440 addresses take 0.13-0.18 ms).  The atomic's return value
// is the block's offset inside the bucket, so every sample already knows its position in the bucket (ch.pos).
__global__ void __launch_bounds__(KEY_THREADS)
tcs_key_kernel(DetGeom g, TcPlan tp, TcChunk ch, const double *__restrict__ p_ra, const double *__restrict__ p_dec,
               int use_smem) {
  extern __shared__ int s_hist[];                                            // [2 n_bkt]
  const int nb2 = 2 * tp.n_bkt;
  const int64_t w0 = (int64_t)blockIdx.x * KEY_THREADS;
  const int64_t seg0 = ch.gb0 / ch.nbps;
  const int lseg0 = (int)((ch.gb0 + w0 / RIFT_TC_NB) / ch.nbps - seg0);
  if (use_smem) {
    for (int i = threadIdx.x; i < nb2; i += KEY_THREADS) s_hist[i] = 0;
    __syncthreads();
  }
  const int64_t w = w0 + threadIdx.x;
  int b = -1;
  if (w < ch.n_batches * RIFT_TC_NB) {
    const int64_t gb = ch.gb0 + w / RIFT_TC_NB;
    const int64_t seg = gb / ch.nbps;
    const int64_t i = (gb % ch.nbps) * RIFT_TC_NB + (w % RIFT_TC_NB);
    if (i < ch.n_per_seg) {
      const int64_t gi = seg * ch.n_per_seg + i;
      double sd, cd, sh, chh;
      sincos(p_dec[gi], &sd, &cd);
      sincos(p_ra[gi] - g.gmst, &sh, &chh);
      const double nx = __dmul_rn(cd, chh), ny = __dmul_rn(cd, sh), nz = sd;
      int32_t shift[2];
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        const double dot =
            __dadd_rn(__dadd_rn(__dmul_rn(g.loc[k][0], nx), __dmul_rn(g.loc[k][1], ny)), __dmul_rn(g.loc[k][2], nz));
        const double dt = -__ddiv_rn(dot, RIFT_C_LIGHT);
        const double x = __ddiv_rn(dt, g.delta_t);
        shift[k] = (int32_t)floor(__dadd_rn(x, 0.5));
      }
      const int dm = tp.dmax[1];
      int d = shift[1] - shift[0];
      d = d < -dm ? -dm : (d > dm ? dm : d);                                 // only samples with invalid angles can be out of range
      b = (int)(seg - seg0) * tp.n_bkt + d + dm;
    }
  }
  const int rel = b - lseg0 * tp.n_bkt;
  const bool loc = use_smem && b >= 0 && rel < nb2;
  int r = 0;
  if (loc) r = atomicAdd(&s_hist[rel], 1);
  else if (b >= 0) r = atomicAdd(ch.count + b, 1);
  if (use_smem) {
    __syncthreads();
    for (int i = threadIdx.x; i < nb2; i += KEY_THREADS) {
      const int c = s_hist[i];
      if (c > 0) s_hist[i] = atomicAdd(ch.count + lseg0 * tp.n_bkt + i, c);
    }
    __syncthreads();
  }
  if (w < ch.n_batches * RIFT_TC_NB) {
    ch.key[w] = b;
    if (b >= 0) ch.pos[w] = loc ? s_hist[rel] + r : r;
  }
}

// pass 2 (one block): batches per bucket, their exclusive prefix, the first batch of every local segment
__global__ void __launch_bounds__(1024) tcs_scan_kernel(TcPlan tp, TcChunk ch) {
  __shared__ int s_warp[32];
  __shared__ int s_carry;
  const int n = ch.n_lseg * tp.n_bkt;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) s_carry = 0;
  __syncthreads();
  for (int i0 = 0; i0 < n; i0 += 1024) {
    const int i = i0 + threadIdx.x;
    const int nb = i < n ? (ch.count[i] + RIFT_TC_NB - 1) / RIFT_TC_NB : 0;
    int v = nb;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, v, o);
      if (lane >= o) v += t;
    }
    if (lane == 31) s_warp[warp] = v;
    __syncthreads();
    if (warp == 0) {
      int t = s_warp[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int u = __shfl_up_sync(0xffffffffu, t, o);
        if (lane >= o) t += u;
      }
      s_warp[lane] = t;
    }
    __syncthreads();
    const int excl = s_carry + (warp ? s_warp[warp - 1] : 0) + v - nb;
    if (i < n) {
      ch.base[i] = excl;
      if (i % tp.n_bkt == 0) ch.seg_begin[i / tp.n_bkt] = excl;
    }
    __syncthreads();
    if (threadIdx.x == 1023) s_carry = excl + nb;
    __syncthreads();
  }
  if (threadIdx.x == 0) ch.seg_begin[ch.n_lseg] = s_carry;
}
}  // namespace

namespace {
// pass 3: sorted slot of every sample = first slot of its bucket + position in the bucket; perm was preset to -1 (padding)
__global__ void __launch_bounds__(256) tcs_fill_kernel(TcChunk ch) {
  const int64_t w = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (w >= ch.n_batches * RIFT_TC_NB) return;
  const int b = ch.key[w];
  if (b < 0) return;
  ch.perm[(int64_t)ch.base[b] * RIFT_TC_NB + ch.pos[w]] = (int32_t)w;
}
}  // namespace

cudaError_t launch_tcs_buckets(const DetGeom &g, const TcPlan &tp, const TcChunk &c, const double *const params[6],
                               cudaStream_t s, int *n_launch) {
  const int64_t n = c.n_batches * RIFT_TC_NB;
  if (n <= 0) return cudaSuccess;
  cudaError_t e = cudaMemsetAsync(c.count, 0, sizeof(int32_t) * (size_t)c.n_lseg * tp.n_bkt, s);
  if (e != cudaSuccess) return e;
  const int use_smem = 2 * tp.n_bkt * (int)sizeof(int) <= 32 * 1024 ? 1 : 0;
  tcs_key_kernel<<<(unsigned)((n + KEY_THREADS - 1) / KEY_THREADS), KEY_THREADS, use_smem ? 2 * tp.n_bkt * sizeof(int) : 0, s>>>(
      g, tp, c, params[0], params[1], use_smem);
  tcs_scan_kernel<<<1, 1024, 0, s>>>(tp, c);
  e = cudaMemsetAsync(c.perm, 0xff, sizeof(int32_t) * (size_t)c.cap_sorted * RIFT_TC_NB, s);
  if (e != cudaSuccess) return e;
  tcs_fill_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(c);
  if (n_launch) *n_launch += 3;
  return cudaGetLastError();
}

cudaError_t launch_geometry_tc(const DetGeom &g, const ModeEntry *modes, const TcPlan &tp, const TcChunk &c,
                               const double *const params[6], const double *U, const double *V, const QuadProg &qp,
                               int32_t *shift_out, cudaStream_t s) {
  const int64_t n = (c.key ? c.cap_sorted : c.n_batches) * RIFT_TC_NB;      // sorted variant: upper bound, trimmed on device
  if (n <= 0) return cudaSuccess;
  const unsigned grid = (unsigned)((n + GEOM_THREADS - 1) / GEOM_THREADS);
  if (tp.n_sub > 1) {
    const size_t uv_bytes = (size_t)2 * tp.K * tp.M * tp.M * sizeof(double2);
    const size_t prog_bytes = quad_smem(qp.n_entries, tp.K, tp.M).total;
    const bool prog = qp.uv != nullptr && prog_bytes <= 96u * 1024u;
    const int stage_uv = uv_bytes <= 96u * 1024u ? 1 : 0;                    // else U, V are read through L1
    const size_t smem = prog ? prog_bytes : (stage_uv ? uv_bytes : 0);
#define RIFT_GEOM_TCX_MS(KT, MS)                                                                                         \
  case MS: {                                                                                                             \
    auto kern = prog ? geometry_tcx_kernel<KT, MS, true> : geometry_tcx_kernel<KT, MS, false>;                           \
    if (smem > 48u * 1024u) {                                                                                            \
      cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);                \
      if (e != cudaSuccess) return e;                                                                                    \
    }                                                                                                                    \
    kern<<<grid, GEOM_THREADS, smem, s>>>(g, modes, tp, c, params[0], params[1], params[2], params[3], params[4],        \
                                          params[5], U, V, qp, shift_out, stage_uv);                                     \
    break;                                                                                                               \
  }
#define RIFT_GEOM_TCX(KT)                                                                                                \
  case KT:                                                                                                               \
    switch (tp.m_sub) {                                                                                                  \
      RIFT_GEOM_TCX_MS(KT, 5) RIFT_GEOM_TCX_MS(KT, 6) RIFT_GEOM_TCX_MS(KT, 7) RIFT_GEOM_TCX_MS(KT, 8)                    \
      default: return cudaErrorInvalidValue;                                                                             \
    }                                                                                                                    \
    break;
    switch (tp.K) {
      RIFT_GEOM_TCX(1) RIFT_GEOM_TCX(2) RIFT_GEOM_TCX(3) RIFT_GEOM_TCX(4) RIFT_GEOM_TCX(5)
      default: return cudaErrorInvalidValue;
    }
#undef RIFT_GEOM_TCX_MS
#undef RIFT_GEOM_TCX
    return cudaGetLastError();
  }
  switch (tp.M) {
    case 1: return launch_geometry_tc_m<1>(g, modes, tp, c, params, U, V, shift_out, grid, s);
    case 2: return launch_geometry_tc_m<2>(g, modes, tp, c, params, U, V, shift_out, grid, s);
    case 3: return launch_geometry_tc_m<3>(g, modes, tp, c, params, U, V, shift_out, grid, s);
    case 4: return launch_geometry_tc_m<4>(g, modes, tp, c, params, U, V, shift_out, grid, s);
    case 5: return launch_geometry_tc_m<5>(g, modes, tp, c, params, U, V, shift_out, grid, s);
    case 6: return launch_geometry_tc_m<6>(g, modes, tp, c, params, U, V, shift_out, grid, s);
    case 7: return launch_geometry_tc_m<7>(g, modes, tp, c, params, U, V, shift_out, grid, s);
    case 8: return launch_geometry_tc_m<8>(g, modes, tp, c, params, U, V, shift_out, grid, s);
    default: return cudaErrorInvalidValue;
  }
}

namespace {
template <typename CT, int MAXM>
cudaError_t launch_geometry_k(const DetGeom &g, const ModeEntry *modes, const Batch &b, const double *const params[6],
                              const double *U, const double *V, const QuadProg &qp, const Workspace &ws, int32_t *shift_out, double *dbg_F,
                              double *dbg_Y, const int32_t *perm, unsigned grid, cudaStream_t s) {
  const size_t uv_bytes = (size_t)2 * g.n_det * g.n_modes * g.n_modes * sizeof(double2);
  const int stage_uv = (MAXM > 16 && uv_bytes <= 96u * 1024u) ? 1 : 0;      // large mode sets: U, V from shared memory
  const size_t prog_bytes = quad_smem(qp.n_entries, g.n_det, g.n_modes).total;
  constexpr bool CAN_PROG = MAXM > 16;
  const bool prog = CAN_PROG && qp.uv != nullptr && prog_bytes <= 96u * 1024u;
  const size_t smem = prog ? prog_bytes : (stage_uv ? uv_bytes : 0);
#define RIFT_GEOM(KT)                                                                                                   \
  case KT: {                                                                                                            \
    auto kern = prog ? geometry_kernel<CT, MAXM, KT, CAN_PROG> : geometry_kernel<CT, MAXM, KT, false>;                  \
    if (smem > 48u * 1024u) {                                                                                           \
      cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);               \
      if (e != cudaSuccess) return e;                                                                                   \
    }                                                                                                                   \
    kern<<<grid, GEOM_THREADS, smem, s>>>(g, modes, b, params[0], params[1], params[2], params[3], params[4], params[5], \
                                          U, V, qp, ws, shift_out, dbg_F, dbg_Y, perm, stage_uv);                       \
    break;                                                                                                              \
  }
  switch (g.n_det) {
    RIFT_GEOM(1) RIFT_GEOM(2) RIFT_GEOM(3) RIFT_GEOM(4) RIFT_GEOM(5) RIFT_GEOM(6) RIFT_GEOM(7) RIFT_GEOM(8)
    default: return cudaErrorInvalidValue;
  }
#undef RIFT_GEOM
  return cudaGetLastError();
}
}  // namespace

cudaError_t launch_geometry(const DetGeom &g, const ModeEntry *modes, const Batch &b, const double *const params[6],
                            const double *U, const double *V, const QuadProg &qp, bool coef_fp32, const Workspace &ws,
                            int32_t *shift_out, double *dbg_F, double *dbg_Y, const int32_t *perm, cudaStream_t s) {
  if (b.n <= 0) return cudaSuccess;
  const unsigned grid = (unsigned)((b.n + GEOM_THREADS - 1) / GEOM_THREADS);
  const bool small = g.n_modes <= 8;
  if (coef_fp32)
    return small ? launch_geometry_k<float2, 8>(g, modes, b, params, U, V, qp, ws, shift_out, dbg_F, dbg_Y, perm, grid, s)
                 : launch_geometry_k<float2, RIFT_MAX_MODES>(g, modes, b, params, U, V, qp, ws, shift_out, dbg_F, dbg_Y, perm,
                                                             grid, s);
  return small ? launch_geometry_k<double2, 8>(g, modes, b, params, U, V, qp, ws, shift_out, dbg_F, dbg_Y, perm, grid, s)
               : launch_geometry_k<double2, RIFT_MAX_MODES>(g, modes, b, params, U, V, qp, ws, shift_out, dbg_F, dbg_Y, perm,
                                                            grid, s);
}

cudaError_t launch_build_quad_uv(const QuadProg &qp, const double *U, const double *V, int32_t P, int32_t K, int32_t M,
                                 double2 *uv_out, cudaStream_t s) {
  const int64_t total = (int64_t)P * qp.n_entries * K;
  if (total <= 0) return cudaSuccess;
  build_quad_uv_kernel<<<(unsigned)((total + 255) / 256), 256, 0, s>>>(qp, reinterpret_cast<const double2 *>(U),
                                                                       reinterpret_cast<const double2 *>(V), P, K, M, uv_out);
  return cudaGetLastError();
}

// Geometry kernel: steps a1-a5 of DESIGN.md section 1, one thread per extrinsic sample, always fp64.
//   a1 F_k = F+ + i Fx from (ra, dec, psi), GMST and the response tensor D_k   (reading G2; F_k of Eq. (D2)-(D3),
//      PAPER.md:763-766)
//   a2 Y_lm = -2Y_lm(iota, -phi_ref) from the per-mode term tables built at create   (reading G3)
//   a3 dt_k = -(r_k . n)/c, s_k = floor(dt_k/delta_t + 1/2), pinned operation order   (reading G4; t_k of Eq. (D2))
//   a4 q = (c^2/4) sum_k [ |F_k|^2 Y^dag U_k Y + Re(F_k^2 Y^T V_k Y) ]               (Eq. (D3))
//   a5 coefficient vector B_{k,lm} = F_k Y_lm, so that Re sum conj(B) Q = sum (B.re Q.re + B.im Q.im)
#include "rift_internal.h"

namespace {

constexpr int GEOM_THREADS = 128;

template <typename CT>
__global__ void __launch_bounds__(GEOM_THREADS)
geometry_kernel(DetGeom g, const ModeEntry *__restrict__ modes, Batch b, const double *__restrict__ p_ra,
                const double *__restrict__ p_dec, const double *__restrict__ p_psi, const double *__restrict__ p_iota,
                const double *__restrict__ p_phi, const double *__restrict__ p_dist, const double *__restrict__ U,
                const double *__restrict__ V, Workspace ws, int32_t *__restrict__ shift_out,
                double *__restrict__ dbg_F, double *__restrict__ dbg_Y, const int32_t *__restrict__ perm) {
  const int64_t w = (int64_t)blockIdx.x * GEOM_THREADS + threadIdx.x;     // workspace slot (sorted position)
  if (w >= b.n) return;
  const int64_t src = perm ? (int64_t)perm[w] : w;                         // chunk-local index of the sample
  if (ws.orig) ws.orig[w] = (int32_t)src;
  const int64_t gi = b.g0 + src;                                           // caller's sample index
  const int32_t point = b.ids[gi / b.n_per_seg];
  const int K = g.n_det, M = g.n_modes;

  const double ra = p_ra[gi], dec = p_dec[gi], psi = p_psi[gi], iota = p_iota[gi], phi = p_phi[gi], dist = p_dist[gi];

  double sd, cd, sh, ch, sp, cp;
  sincos(dec, &sd, &cd);
  sincos(ra - g.gmst, &sh, &ch);           // ch = cos(ra-gmst) = cos(gha), sh = sin(ra-gmst) = -sin(gha)
  sincos(psi, &sp, &cp);

  // ---- a3: delays and integer shifts, every operation individually rounded (no FMA contraction)
  const double nx = __dmul_rn(cd, ch), ny = __dmul_rn(cd, sh), nz = sd;
  int32_t *my_shift = ws.shift + w * K;
  for (int k = 0; k < K; ++k) {
    const double dot = __dadd_rn(__dadd_rn(__dmul_rn(g.loc[k][0], nx), __dmul_rn(g.loc[k][1], ny)),
                                 __dmul_rn(g.loc[k][2], nz));
    const double dt = -__ddiv_rn(dot, RIFT_C_LIGHT);
    const double x = __ddiv_rn(dt, g.delta_t);
    const int32_t s = (int32_t)floor(__dadd_rn(x, 0.5));
    my_shift[k] = s;
    if (shift_out) shift_out[gi * K + k] = s;
  }

  // ---- a1: antenna factors
  const double sg = -sh, cg = ch;          // sin, cos of the Greenwich hour angle gmst - ra
  const double X[3] = {-cp * sg - sp * cg * sd, -cp * cg + sp * sg * sd, sp * cd};
  const double Yv[3] = {sp * sg - cp * cg * sd, sp * cg + cp * sg * sd, cp * cd};
  double Fre[RIFT_MAX_DET], Fim[RIFT_MAX_DET];
#pragma unroll
  for (int k = 0; k < RIFT_MAX_DET; ++k) {
    if (k < K) {
      const double *D = g.resp[k];
      double xdx = 0, ydy = 0, xdy = 0, ydx = 0;
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
          const double d = D[3 * i + j];
          xdx += X[i] * d * X[j];
          ydy += Yv[i] * d * Yv[j];
          xdy += X[i] * d * Yv[j];
          ydx += Yv[i] * d * X[j];
        }
      Fre[k] = xdx - ydy;
      Fim[k] = xdy + ydx;
      if (dbg_F) {
        dbg_F[(gi * K + k) * 2] = Fre[k];
        dbg_F[(gi * K + k) * 2 + 1] = Fim[k];
      }
    }
  }

  // ---- a2: harmonics.  powers of cos(iota/2), sin(iota/2); e^{-i m phi} by angle addition
  double pc[17], ps[17], cm[9], sm[9];
  {
    double shalf, chalf;
    sincos(0.5 * iota, &shalf, &chalf);
    pc[0] = ps[0] = 1.0;
    const int np = 2 * g.l_max;
    for (int i = 1; i <= 16; ++i) {
      pc[i] = (i <= np) ? pc[i - 1] * chalf : 0.0;
      ps[i] = (i <= np) ? ps[i - 1] * shalf : 0.0;
    }
    double s1, c1;
    sincos(phi, &s1, &c1);
    cm[0] = 1.0;
    sm[0] = 0.0;
    for (int i = 1; i <= 8; ++i) {
      cm[i] = cm[i - 1] * c1 - sm[i - 1] * s1;
      sm[i] = sm[i - 1] * c1 + cm[i - 1] * s1;
    }
  }
  double Yre[RIFT_MAX_MODES], Yim[RIFT_MAX_MODES];
  for (int a = 0; a < M; ++a) {
    const ModeEntry &e = modes[a];
    double amp = 0.0;
    for (int t = 0; t < e.n_terms; ++t) amp += e.coef[t] * pc[e.pc[t]] * ps[e.ps[t]];
    const int am = e.m < 0 ? -e.m : e.m;
    // e^{i m (-phi)} = cos(m phi) - i sin(m phi)
    Yre[a] = amp * cm[am];
    Yim[a] = (e.m < 0) ? amp * sm[am] : -amp * sm[am];
    if (dbg_Y) {
      dbg_Y[(gi * M + a) * 2] = Yre[a];
      dbg_Y[(gi * M + a) * 2 + 1] = Yim[a];
    }
  }

  // ---- a5: coefficient vectors B = F_k Y_lm
  const bool bad = !(dist > 0.0) || isnan(ra) || isnan(dec) || isnan(psi) || isnan(iota) || isnan(phi);
  const double c = bad ? __longlong_as_double(0x7ff8000000000000LL) : g.d_ref / dist;
  ws.scale_c[w] = c;
  {
    CT *out = reinterpret_cast<CT *>(reinterpret_cast<decltype(CT::x) *>(ws.coef) + w * ws.coef_stride);
    for (int k = 0; k < K; ++k)
      for (int a = 0; a < M; ++a) {
        CT v;
        v.x = Fre[k] * Yre[a] - Fim[k] * Yim[a];
        v.y = Fre[k] * Yim[a] + Fim[k] * Yre[a];
        out[k * M + a] = v;
      }
  }

  // ---- a4: quadratic term; U Hermitian, V symmetric: diagonal + 2 * strict upper triangle
  double q = 0.0;
  for (int k = 0; k < K; ++k) {
    const double2 *Uk = reinterpret_cast<const double2 *>(U) + ((int64_t)point * K + k) * M * M;
    const double2 *Vk = reinterpret_cast<const double2 *>(V) + ((int64_t)point * K + k) * M * M;
    double yuy = 0.0, yvy_re = 0.0, yvy_im = 0.0;
    for (int a = 0; a < M; ++a) {
      const double ar = Yre[a], ai = Yim[a];
      {
        const double2 u = Uk[a * M + a], v = Vk[a * M + a];
        yuy += u.x * (ar * ar + ai * ai);
        const double y2r = ar * ar - ai * ai, y2i = 2.0 * ar * ai;
        yvy_re += v.x * y2r - v.y * y2i;
        yvy_im += v.x * y2i + v.y * y2r;
      }
      for (int bb = a + 1; bb < M; ++bb) {
        const double br = Yre[bb], bi = Yim[bb];
        const double2 u = Uk[a * M + bb], v = Vk[a * M + bb];
        // conj(Y_a) Y_b and Y_a Y_b
        const double cr = ar * br + ai * bi, ci = ar * bi - ai * br;
        const double pr = ar * br - ai * bi, pi = ar * bi + ai * br;
        yuy += 2.0 * (u.x * cr - u.y * ci);
        yvy_re += 2.0 * (v.x * pr - v.y * pi);
        yvy_im += 2.0 * (v.x * pi + v.y * pr);
      }
    }
    const double f2 = Fre[k] * Fre[k] + Fim[k] * Fim[k];
    const double f2r = Fre[k] * Fre[k] - Fim[k] * Fim[k], f2i = 2.0 * Fre[k] * Fim[k];
    q += f2 * yuy + (f2r * yvy_re - f2i * yvy_im);
  }
  ws.quad[w] = 0.25 * c * c * q;
}

}  // namespace

cudaError_t launch_geometry(const DetGeom &g, const ModeEntry *modes, const Batch &b, const double *const params[6],
                            const double *U, const double *V, bool coef_fp32, const Workspace &ws,
                            int32_t *shift_out, double *dbg_F, double *dbg_Y, const int32_t *perm, cudaStream_t s) {
  if (b.n <= 0) return cudaSuccess;
  const int64_t n = b.n;
  const unsigned grid = (unsigned)((n + GEOM_THREADS - 1) / GEOM_THREADS);
  if (coef_fp32)
    geometry_kernel<float2><<<grid, GEOM_THREADS, 0, s>>>(g, modes, b, params[0], params[1], params[2], params[3],
                                                           params[4], params[5], U, V, ws, shift_out, dbg_F, dbg_Y, perm);
  else
    geometry_kernel<double2><<<grid, GEOM_THREADS, 0, s>>>(g, modes, b, params[0], params[1], params[2], params[3],
                                                            params[4], params[5], U, V, ws, shift_out, dbg_F, dbg_Y, perm);
  return cudaGetLastError();
}

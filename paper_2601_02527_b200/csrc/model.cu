// model.cu -- host side: kernel description -> block-diagonal state-space model in block units.
//
// Sums of kernels stack block-diagonally (App. C.1, Eq. C2-C4); the product
// Matern-3/2 x cos(j w_p tau) is the Kronecker form of App. C.2 (Eq. C6-C9).
// SHO: App. B.  Matern forms: DESIGN.md reading R10 (the paper cites, does not print).
// Every block is written in its own units (time T_b, amplitude sigma_b) so that the constants the
// device sees are O(1); the per-instrument coupling c_qb = sigma_b T_b / tau_q carries the units.
#include <math.h>
#include <string.h>

#include "common.h"

typedef long double ld;

// scaled modified Bessel function exp(-x) I_j(x), power series (x = 1/ell_p^2 is O(1))
static ld bessel_ie(int j, ld x) {
  ld term = 1.0L;
  for (int m = 1; m <= j; ++m) term *= (x / 2) / m;
  ld sum = term;
  for (int m = 1; m < 80; ++m) {
    term *= (x / 2) * (x / 2) / ((ld)m * (ld)(m + j));
    sum += term;
    if (term < 1e-25L * sum) break;
  }
  return sum * expl(-x);
}

static void set_block_common(BlockConst& B, int family, int dim, const ld* F, const ld* W, const ld* H,
                             const ld* Pinf) {
  B.family = family;
  B.dim = dim;
  const int m = dim + 1;
  // augmented F~'' and W~'' (Eq. 3.4-3.6)
  ld Ft[SG_BE * SG_BE] = {0}, Wt[SG_BE * SG_BE] = {0};
  for (int i = 0; i < dim; ++i)
    for (int j = 0; j < dim; ++j) {
      Ft[i * m + j] = F[i * dim + j];
      Wt[i * m + j] = W[i * dim + j];
    }
  for (int j = 0; j < dim; ++j) Ft[dim * m + j] = H[j];
  ld rho = 0;
  for (int i = 0; i < m; ++i) {
    ld s = 0;
    for (int j = 0; j < m; ++j) s += fabsl(Ft[i * m + j]);
    if (s > rho) rho = s;
  }
  B.rho = (double)rho;
  for (int i = 0; i < dim * dim; ++i) B.pinf[i] = (double)Pinf[i];
  // Taylor coefficients: Phi~(h) = sum_k F~^k h^k / k!,  Q~(h) = sum_{k>=1} Gamma_k h^k / k!
  // (Gamma_1 = W~, Gamma_{k+1} = F~ Gamma_k + Gamma_k F~^T: term-by-term integration of
  // int_0^h e^{F~ s} W~ e^{F~^T s} ds, the integral behind Eq. 2.19 / 3.10).
  ld Ak[SG_BE * SG_BE] = {0}, Gk[SG_BE * SG_BE] = {0}, T1[SG_BE * SG_BE];
  for (int i = 0; i < m; ++i) Ak[i * m + i] = 1;
  memset(B.tayA, 0, sizeof(B.tayA));
  memset(B.tayQ, 0, sizeof(B.tayQ));
  ld fact = 1;
  for (int k = 0; k <= SG_KT; ++k) {
    if (k > 0) fact *= k;
    for (int i = 0; i < m; ++i)
      for (int j = 0; j < m; ++j) {
        B.tayA[k][i * SG_BE + j] = (double)(Ak[i * m + j] / fact);
        B.tayQ[k][i * SG_BE + j] = (double)(Gk[i * m + j] / fact);
      }
    // next power / next Gamma
    for (int i = 0; i < m; ++i)
      for (int j = 0; j < m; ++j) {
        ld s = 0;
        for (int l = 0; l < m; ++l) s += Ft[i * m + l] * Ak[l * m + j];
        T1[i * m + j] = s;
      }
    memcpy(Ak, T1, sizeof(T1));
    if (k == 0) {
      memcpy(Gk, Wt, sizeof(Wt));
    } else {
      for (int i = 0; i < m; ++i)
        for (int j = 0; j < m; ++j) {
          ld s = 0;
          for (int l = 0; l < m; ++l) s += Ft[i * m + l] * Gk[l * m + j] + Gk[i * m + l] * Ft[j * m + l];
          T1[i * m + j] = s;
        }
      memcpy(Gk, T1, sizeof(T1));
    }
  }
}

static void make_m32(BlockConst& B, ld lambda) {
  const ld F[4] = {0, 1, -1, -2}, W[4] = {0, 0, 0, 4}, H[2] = {1, 0}, P[4] = {1, 0, 0, 1};
  set_block_common(B, BLK_M32, 2, F, W, H, P);
  B.inv_T = (double)lambda;
  B.a = B.b = 0;
  B.sho_case = 0;
}
static void make_m52(BlockConst& B, ld lambda) {
  const ld F[9] = {0, 1, 0, 0, 0, 1, -1, -3, -3};
  const ld W[9] = {0, 0, 0, 0, 0, 0, 0, 0, 16.0L / 3};
  const ld H[3] = {1, 0, 0};
  const ld P[9] = {1, 0, -1.0L / 3, 0, 1.0L / 3, 0, -1.0L / 3, 0, 1};
  set_block_common(B, BLK_M52, 3, F, W, H, P);
  B.inv_T = (double)lambda;
  B.a = B.b = 0;
  B.sho_case = 0;
}
static void make_sho(BlockConst& B, ld w0, ld Q) {
  const ld F[4] = {0, 1, -1, -1 / Q}, W[4] = {0, 0, 0, 2 / Q}, H[2] = {1, 0}, P[4] = {1, 0, 0, 1};
  set_block_common(B, BLK_SHO, 2, F, W, H, P);
  B.inv_T = (double)w0;
  ld a = 1 / (2 * Q);
  B.a = (double)a;
  if (Q > 0.5L) { B.sho_case = 0; B.b = (double)sqrtl(1 - a * a); }
  else if (Q == 0.5L) { B.sho_case = 1; B.b = 0; }
  else { B.sho_case = 2; B.b = (double)sqrtl(a * a - 1); }
}
static void make_m32rot(BlockConst& B, ld lambda, ld omega) {
  // state index 2a + c, a = Matern index, c = rotation index (Kronecker sum C6)
  const ld w = omega / lambda;
  ld F[16] = {0}, W[16] = {0}, P[16] = {0};
  const ld FM[4] = {0, 1, -1, -2};
  const ld FR[4] = {0, -w, w, 0};
  for (int a = 0; a < 2; ++a)
    for (int c = 0; c < 2; ++c)
      for (int a2 = 0; a2 < 2; ++a2)
        for (int c2 = 0; c2 < 2; ++c2)
          F[(2 * a + c) * 4 + 2 * a2 + c2] = FM[a * 2 + a2] * (c == c2) + (a == a2) * FR[c * 2 + c2];
  W[2 * 4 + 2] = 4; W[3 * 4 + 3] = 4; // W_M32 (x) Pinf_rot (C8)
  for (int i = 0; i < 4; ++i) P[i * 4 + i] = 1;
  const ld H[4] = {1, 0, 0, 0};
  set_block_common(B, BLK_M32ROT, 4, F, W, H, P);
  B.inv_T = (double)lambda;
  B.a = 0;
  B.b = (double)w;
  B.sho_case = 0;
}

int sg_build_model(smolgp_ctx* ctx, const smolgp_kernel* kern, int n_inst, const double* tau, int instant, ModelDev* M) {
  if (!kern || kern->n_comp <= 0 || !kern->comp) { ctx->err = "kernel: no components"; return SMOLGP_EINVAL; }
  if (n_inst < 1 || n_inst > SG_MAXINST) { ctx->err = "n_inst out of range"; return SMOLGP_EUNSUPPORTED; }
  memset(M, 0, sizeof(*M));
  int nb = 0, d = 0;
  ld sig[SG_MAXBLK];
  uint32_t mask[SG_MAXBLK];
  for (int c = 0; c < kern->n_comp; ++c) {
    const smolgp_component& k = kern->comp[c];
    if (!(k.sigma > 0) || !(k.p0 > 0) || !isfinite(k.sigma) || !isfinite(k.p0)) { ctx->err = "kernel: sigma and p0 must be > 0"; return SMOLGP_EINVAL; }
    int need = (k.family == SMOLGP_MATERN32_X_PERIODIC) ? 1 + (k.order > 0 ? k.order : 0) : 1;
    if (nb + need > SG_MAXBLK) { ctx->err = "kernel: too many blocks"; return SMOLGP_EUNSUPPORTED; }
    switch (k.family) {
      case SMOLGP_MATERN32: make_m32(M->blk[nb], sqrtl(3.0L) / k.p0); sig[nb] = k.sigma; mask[nb] = k.inst_mask; ++nb; break;
      case SMOLGP_MATERN52: make_m52(M->blk[nb], sqrtl(5.0L) / k.p0); sig[nb] = k.sigma; mask[nb] = k.inst_mask; ++nb; break;
      case SMOLGP_SHO:
        if (!(k.p1 > 0)) { ctx->err = "SHO: Q must be > 0"; return SMOLGP_EINVAL; }
        make_sho(M->blk[nb], k.p0, k.p1); sig[nb] = k.sigma; mask[nb] = k.inst_mask; ++nb; break;
      case SMOLGP_MATERN32_X_PERIODIC: {
        if (!(k.p1 > 0) || !(k.p2 > 0) || k.order < 0) { ctx->err = "periodic: period, ell_p > 0, order >= 0"; return SMOLGP_EINVAL; }
        const ld lam = sqrtl(3.0L) / k.p0, wp = 2 * 3.14159265358979323846264338327950288L / k.p1;
        const ld x = 1.0L / ((ld)k.p2 * k.p2);
        for (int j = 0; j <= k.order; ++j) { // reading R11: q_0^2 = I_0 e^-x, q_j^2 = 2 I_j e^-x
          ld q2 = (j == 0 ? 1.0L : 2.0L) * bessel_ie(j, x);
          if (j == 0) make_m32(M->blk[nb], lam); else make_m32rot(M->blk[nb], lam, j * wp);
          sig[nb] = k.sigma * sqrtl(q2); mask[nb] = k.inst_mask; ++nb;
        }
        break;
      }
      default: ctx->err = "kernel: unknown family"; return SMOLGP_EUNSUPPORTED;
    }
  }
  int off = 0;
  for (int b = 0; b < nb; ++b) { M->blk[b].off = d; d += M->blk[b].dim; M->disc_off[b] = off; off += disc_block_size(M->blk[b].dim); }
  if (d + n_inst > SMOLGP_MAX_DIM) { ctx->err = "augmented state dimension above SMOLGP_MAX_DIM"; return SMOLGP_EUNSUPPORTED; }
  M->n = d + n_inst; M->d = d; M->n_inst = n_inst; M->nblk = nb; M->disc_stride = off; M->instant = instant;
  for (int q = 0; q < n_inst; ++q) {
    M->tau[q] = tau[q];
    for (int b = 0; b < nb; ++b)
      // integrated data: z_q/tau_q gathers sigma_b T_b I''_b (I'' = int x''_0 dt'').  Instantaneous data (section 2): z_q is
      // SET to H_q x = sum_b sigma_b x''_{b,0} at its sample, through the same coupling with the record's integral
      // rows replaced by H Phi (disc.cu), so the coupling is sigma_b / tau_q
      M->cz[q][b] = ((mask[b] >> q) & 1u) ? (double)(instant ? sig[b] / (ld)tau[q] : sig[b] / ((ld)M->blk[b].inv_T * (ld)tau[q])) : 0.0;
  }
  for (int b = 0; b < nb; ++b) { M->bsig[b] = (double)sig[b]; M->bmask[b] = mask[b]; }
  const int n = M->n;
  for (int b = 0; b < nb; ++b)
    for (int i = 0; i < M->blk[b].dim; ++i)
      for (int j = 0; j < M->blk[b].dim; ++j)
        M->p0[(M->blk[b].off + i) * n + M->blk[b].off + j] = M->blk[b].pinf[i * M->blk[b].dim + j];
  return SMOLGP_OK;
}

// disc.cu -- step a2: per-event discretisation of every block of the augmented model.
//
// For a step of length Delta the augmented block [x_b; I_b] (I_b = int H_b x_b dt, Eq. 3.3-3.6,
// P:365-381) needs Phi~ = exp(F~ Delta) = [Phi 0; Phi-bar 1] (Eq. 3.7) and
// Q~ = int_0^Delta Phi~(s) L~ Qc L~^T Phi~(s)^T ds (Eq. 3.10).  The paper offers the
// Van Loan block exponential (Eq. 3.9, B13) and warns that it is unstable over long gaps (P:193,
// P:407) -- and the printed closed forms (B12, B19, B20) cancel catastrophically for short steps.
// Here, per block and in the block's own O(1) units:
//   1. h = Delta'' / 2^s with rho h <= 1/4: Phi~(h), Q~(h) by their Taylor series (Horner, the
//      coefficients F~^k/k!, Gamma_k/k! are host-built constants) -- exact to rounding, no cancellation;
//   2. s doublings  Q~(2h) = Q~(h) + Phi~(h) Q~(h) Phi~(h)^T,  Phi-bar(2h) = Phi-bar(h) (Phi(h) + I)
//      (sums of PSD terms; no growing exponential ever appears), where Phi(h) at every level is the
//      CLOSED FORM of the family (B10, and its Matern analogues) instead of a repeated
//      square, so the error grows like s eps, not 2^s eps;
//   3. Phi(Delta) itself from the closed form.
// One thread per (event, block), blocks along grid.y; output record layout in common.h.
#include "common.h"

template <int DB>
__device__ __forceinline__ void phi_closed(const BlockConst& B, double h, double (&P)[DB][DB]);

template <>
__device__ __forceinline__ void phi_closed<2>(const BlockConst& B, double h, double (&P)[2][2]) {
  if (B.family == BLK_M32 || (B.family == BLK_SHO && B.sho_case == 1)) {
    // repeated root -1:  e^{-h} (I + h (F + I)),  F + I = [1 1; -1 -1]   (B10 with Q = 1/2)
    const double e = exp(-h);
    P[0][0] = e * (1.0 + h); P[0][1] = e * h; P[1][0] = -e * h; P[1][1] = e * (1.0 - h);
  } else if (B.sho_case == 0) {
    // underdamped: e^{-a h} [cos(b h) I + sin(b h)/b (F + a I)],  F + a I = [a 1; -1 -a]   (B10)
    const double e = exp(-B.a * h);
    double sn, cs;
    sincos(B.b * h, &sn, &cs);
    const double sb = sn / B.b;
    P[0][0] = e * (cs + B.a * sb); P[0][1] = e * sb; P[1][0] = -e * sb; P[1][1] = e * (cs - B.a * sb);
  } else {
    // overdamped: cos -> cosh, sin/b -> sinh/beta, with the decaying exponentials combined
    const double e1 = exp(-(B.a - B.b) * h), e2 = exp(-(B.a + B.b) * h);
    const double ch = 0.5 * (e1 + e2), sb = 0.5 * (e1 - e2) / B.b;
    P[0][0] = ch + B.a * sb; P[0][1] = sb; P[1][0] = -sb; P[1][1] = ch - B.a * sb;
  }
}
template <>
__device__ __forceinline__ void phi_closed<3>(const BlockConst& B, double h, double (&P)[3][3]) {
  // triple root -1:  e^{-h} (I + h N + h^2/2 N^2),  N = F + I = [1 1 0; 0 1 1; -1 -3 -2]
  const double e = exp(-h), h2 = 0.5 * h * h;
  // N^2 = [1 2 1; -1 -2 -1; 1 2 1]
  P[0][0] = e * (1.0 + h + h2);  P[0][1] = e * (h + 2.0 * h2);        P[0][2] = e * h2;
  P[1][0] = e * (-h2);           P[1][1] = e * (1.0 + h - 2.0 * h2);  P[1][2] = e * (h - h2);
  P[2][0] = e * (-h + h2);       P[2][1] = e * (-3.0 * h + 2.0 * h2); P[2][2] = e * (1.0 - 2.0 * h + h2);
}
template <>
__device__ __forceinline__ void phi_closed<4>(const BlockConst& B, double h, double (&P)[4][4]) {
  // Phi_M32(h) (x) R(omega h)   (C7: the transition of a product is the Kronecker product)
  const double e = exp(-h);
  const double M[2][2] = {{e * (1.0 + h), e * h}, {-e * h, e * (1.0 - h)}};
  double sn, cs;
  sincos(B.b * h, &sn, &cs);
  const double R[2][2] = {{cs, -sn}, {sn, cs}};
#pragma unroll
  for (int a = 0; a < 2; ++a)
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
      for (int a2 = 0; a2 < 2; ++a2)
#pragma unroll
        for (int c2 = 0; c2 < 2; ++c2) P[2 * a + c][2 * a2 + c2] = M[a][a2] * R[c][c2];
}

template <int DB>
__device__ void disc_block(const BlockConst& B, double dts, int instant, int sqrt_form, double* __restrict__ out) {
  constexpr int M = DB + 1;
  double h = dts;
  int s = 0;
  {
    double x = B.rho * dts;
    while (x > 0.25 && s < 64) { x *= 0.5; h *= 0.5; ++s; }
  }
  // Taylor order.  The slowest-starting entry of Q~ (the integral's own variance) begins at order
  // kmin = 2 DB + 1 in h; keep terms until they fall below 2^-58 of THAT leading term, so that every
  // entry keeps full relative accuracy: x^j kmin! / (kmin + j)! < 2^-58 with x = rho h <= 1/4.
  int kt = 2 * DB + 1;
  {
    const double x = B.rho * h;
    double rel = 1.0;
    while (rel > 3.5e-18 && kt < SG_KT) { ++kt; rel *= x / (double)kt; }
  }
  // Horner only for what has no cheap closed form: the integral row Phi-bar (row DB of Phi~) and the lower triangle of
  // the symmetric Q~ (DB + M (M + 1) / 2 series instead of 2 M^2); Phi(h) itself is the family's closed form, the last
  // column of Phi~ is (0, ..., 0, 1)
  double A[M][M], Q[M][M];
  {
    double P[DB][DB];
    phi_closed<DB>(B, h, P);
#pragma unroll
    for (int i = 0; i < DB; ++i) {
#pragma unroll
      for (int j = 0; j < DB; ++j) A[i][j] = P[i][j];
      A[i][DB] = 0.0;
    }
    A[DB][DB] = 1.0;
  }
#pragma unroll
  for (int j = 0; j < DB; ++j) A[DB][j] = B.tayA[kt][DB * SG_BE + j];
#pragma unroll
  for (int i = 0; i < M; ++i)
#pragma unroll
    for (int j = 0; j <= i; ++j) Q[i][j] = B.tayQ[kt][i * SG_BE + j];
  for (int k = kt - 1; k >= 0; --k) {
#pragma unroll
    for (int j = 0; j < DB; ++j) A[DB][j] = fma(A[DB][j], h, B.tayA[k][DB * SG_BE + j]);
#pragma unroll
    for (int i = 0; i < M; ++i)
#pragma unroll
      for (int j = 0; j <= i; ++j) Q[i][j] = fma(Q[i][j], h, B.tayQ[k][i * SG_BE + j]);
  }
#pragma unroll
  for (int i = 0; i < M; ++i)
#pragma unroll
    for (int j = i + 1; j < M; ++j) Q[i][j] = Q[j][i];
  for (int lev = 0; lev < s; ++lev) {
    if (lev > 0) {
      double P[DB][DB];
      phi_closed<DB>(B, h, P);
#pragma unroll
      for (int i = 0; i < DB; ++i)
#pragma unroll
        for (int j = 0; j < DB; ++j) A[i][j] = P[i][j];
    }
    double T[M][M];
#pragma unroll
    for (int i = 0; i < M; ++i)
#pragma unroll
      for (int j = 0; j < M; ++j) {
        double acc = 0.0;
#pragma unroll
        for (int l = 0; l < M; ++l) acc = fma(A[i][l], Q[l][j], acc);
        T[i][j] = acc;
      }
#pragma unroll
    for (int i = 0; i < M; ++i)
#pragma unroll
      for (int j = 0; j <= i; ++j) {
        double acc = Q[i][j];
#pragma unroll
        for (int l = 0; l < M; ++l) acc = fma(T[i][l], A[j][l], acc);
        Q[i][j] = acc;
      }
#pragma unroll
    for (int i = 0; i < M; ++i)
#pragma unroll
      for (int j = i + 1; j < M; ++j) Q[i][j] = Q[j][i];
    double pb[DB];
#pragma unroll
    for (int c = 0; c < DB; ++c) {
      double acc = A[DB][c];
#pragma unroll
      for (int l = 0; l < DB; ++l) acc = fma(A[DB][l], A[l][c], acc);
      pb[c] = acc;
    }
#pragma unroll
    for (int c = 0; c < DB; ++c) A[DB][c] = pb[c];
    h *= 2.0;
  }
  if (s > 0) {
    double P[DB][DB];
    phi_closed<DB>(B, dts, P);
#pragma unroll
    for (int i = 0; i < DB; ++i)
#pragma unroll
      for (int j = 0; j < DB; ++j) A[i][j] = P[i][j];
  }
  if (sqrt_form) {
    // square-root form (chunk_sqrt.cuh): the record carries L with L L^T = Q~ instead of Q~.  Lower Cholesky factor
    // of a positive SEMI-definite matrix: a pivot that rounding has driven to <= 2^-44 of its diagonal entry gives a
    // zero column (Q~ = 0 at a zero step; for instantaneous data the extra state is a copy of x_0, so only the
    // DB x DB part is factored and the extra row of the factor is row 0 of L_xx)
    const int mm = instant ? DB : M;
#pragma unroll
    for (int j = 0; j < M; ++j) {
      if (j >= mm) break;
      double p = Q[j][j];
#pragma unroll
      for (int k = 0; k < j; ++k) p = fma(-Q[j][k], Q[j][k], p);
      const bool ok = p > Q[j][j] * 5.7e-14;
      const double r = ok ? sqrt(p) : 0.0, rr = ok ? 1.0 / r : 0.0;
#pragma unroll
      for (int i = j + 1; i < M; ++i) {
        double a = Q[i][j];
#pragma unroll
        for (int k = 0; k < j; ++k) a = fma(-Q[i][k], Q[j][k], a);
        Q[i][j] = (i < mm) ? a * rr : Q[i][j];
      }
      Q[j][j] = r;
#pragma unroll
      for (int i = 0; i < j; ++i) Q[i][j] = 0.0;
    }
  }
  // record: Phi | phibar | Qxx | q12 | q22   (square-root form: Phi | phibar | Lxx | Lzx | Lzz)
#pragma unroll
  for (int i = 0; i < DB; ++i)
#pragma unroll
    for (int j = 0; j < DB; ++j) { out[i * DB + j] = A[i][j]; out[DB * DB + DB + i * DB + j] = Q[i][j]; }
  if (instant) {
    // instantaneous data (paper section 2): the extra state of the block is not its integral but its
    // latent after the step, H'' x'' = x''_0: row 0 of Phi, Cov(x'', x''_0) = column 0 of Q, Var(x''_0) = Q_00.  The
    // chunk kernels then carry z_q = H_q x at each sample with their unchanged arithmetic (z_q is idle, i.e.
    // zero, before its sample, so the "+ z_q" of the integral row adds nothing).
#pragma unroll
    for (int j = 0; j < DB; ++j) { out[DB * DB + j] = A[0][j]; out[2 * DB * DB + DB + j] = sqrt_form ? Q[0][j] : Q[j][0]; }
    out[2 * DB * DB + 2 * DB] = sqrt_form ? 0.0 : Q[0][0];
    return;
  }
#pragma unroll
  for (int j = 0; j < DB; ++j) { out[DB * DB + j] = A[DB][j]; out[2 * DB * DB + DB + j] = Q[DB][j]; }
  out[2 * DB * DB + 2 * DB] = Q[DB][DB];
}

// blockIdx.y = block of the model: every thread of a CTA works on the same block, so the Taylor
// coefficients and closed-form constants are warp-uniform loads and the family switch does not diverge
__global__ void __launch_bounds__(128) k_disc(const ModelDev* __restrict__ Mp, const double* __restrict__ dt, int64_t K,
                                              double* __restrict__ disc) {
  extern __shared__ double stage[]; // [128][bs]: each thread's record, then written out in coalesced runs
  const int b = blockIdx.y;
  const int64_t k0 = (int64_t)blockIdx.x * blockDim.x, k = k0 + threadIdx.x;
  const BlockConst& B = Mp->blk[b];
  const int bs = 2 * B.dim * B.dim + 2 * B.dim + 1; // odd: conflict-free per-thread rows
  if (k < K) {
    const double dts = dt[k] * B.inv_T;
    double* out = stage + threadIdx.x * bs;
    switch (B.dim) {
      case 2: disc_block<2>(B, dts, Mp->instant, Mp->sqrt_form, out); break;
      case 3: disc_block<3>(B, dts, Mp->instant, Mp->sqrt_form, out); break;
      default: disc_block<4>(B, dts, Mp->instant, Mp->sqrt_form, out); break;
    }
  }
  __syncthreads();
  const int64_t nev = (K - k0 < blockDim.x) ? (K - k0) : blockDim.x;
  const int stride = Mp->disc_stride, off = Mp->disc_off[b];
  const float rbs = 1.0f / (float)bs;
  for (int e = threadIdx.x; e < (int)nev * bs; e += blockDim.x) {
    const int ev = __float2int_rz(((float)e + 0.5f) * rbs), j = e - ev * bs;
    disc[(k0 + ev) * (int64_t)stride + off + j] = stage[e];
  }
}

int sg_launch_disc(smolgp_ctx* ctx, const ModelDev* d_model, const ModelDev* h_model, const double* dt,
                   int64_t K, double* disc) {
  dim3 grid((unsigned)((K + 127) / 128), (unsigned)h_model->nblk);
  sg_launch_begin(ctx, KID_DISC);
  k_disc<<<grid, 128, 128 * (2 * SG_MAXBD * SG_MAXBD + 2 * SG_MAXBD + 1) * sizeof(double), ctx->stream>>>(d_model, dt, K, disc);
  sg_launch_end(ctx);
  SG_CUDA(ctx, cudaGetLastError());
  return SMOLGP_OK;
}

/* mapl_oracle.c -- TEST INFRASTRUCTURE, not the product.
 *
 * Plain, slow, fp64 CPU statement of what the MAPL boundary codec computes
 * (arxiv/paper_2606_05484; citations "P:NN" are /root/reference/PAPER.md line NN).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call this.  It shares no code with the CUDA path (paper_2606_05484_b200/csrc).
 *
 * Conventions: row-major, row-vector form.  H,Hhat,g,dH are [N,d]; U is [d,r];
 * Z,Zhat,gz are [N,r]; codebooks C are [L,K,r]; anchor factors A [V,ra], B [ra,d];
 * tok is int32 [N].  All floating point is double.  Loops are the textbook definition:
 * no blocking, no fusion, no reordering; OpenMP only splits INDEPENDENT outputs
 * (tokens or output rows), never a reduction, so results do not depend on thread count.
 *
 * Pins (tests/test_oracle_*.py): every function below is checked against closed forms,
 * invariants, finite differences, brute force or a library routine; none is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int mapl_oracle_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ---------------------------------------------------------------- projection (Eq. 1)
 * Z = (H - As[tok] Bs) U.  The hot path takes h as the already-centred residual
 * (north_star: z = U^T h; reading S6), i.e. As == NULL.  The centring term of
 * Eq. 1 is kept behind that flag.                                                        */
void mapl_oracle_project(int64_t N, int d, int r, const double* H, const double* U,
                         const int32_t* tok, const double* As, const double* Bs, int ras,
                         double* Z) {
#pragma omp parallel for schedule(static)
  for (int64_t n = 0; n < N; ++n) {
    for (int j = 0; j < r; ++j) Z[n * r + j] = 0.0;
    for (int i = 0; i < d; ++i) {
      double x = H[n * d + i];
      if (As) {                       /* x - (As[tok_n,:] . Bs[:,i]) */
        double a = 0.0;
        for (int q = 0; q < ras; ++q) a += As[(int64_t)tok[n] * ras + q] * Bs[(int64_t)q * d + i];
        x -= a;
      }
      for (int j = 0; j < r; ++j) Z[n * r + j] += x * U[(int64_t)i * r + j];
    }
  }
}

/* ---------------------------------------------------------------- residual VQ (Sec. 3.5)
 * "Each stage quantizes the residual error from the previous round": rho_0 = z; for each
 * level l: k* = argmin_k sum_j (rho_j - C[l,k,j])^2 (direct form; lowest k on ties, reading
 * S4), rho <- rho - C[l,k*,:].  Zhat = sum_l C[l,codes_l,:].
 * d1/d2 [N,L] receive the smallest and second smallest squared distance (for the near-tie
 * rule, reading S5).  forced [N,L] (may be NULL): an entry >= 0 replaces the argmin at that
 * (token, level) -- used only to follow an admissible near-tie choice (S5).                */
void mapl_oracle_rvq(int64_t N, int r, int L, int K, const double* Z, const double* C,
                     const int32_t* forced, int32_t* codes, double* Zhat, double* rho_out,
                     double* d1, double* d2) {
#pragma omp parallel
  {
    double* rho = (double*)malloc(sizeof(double) * (size_t)r);
#pragma omp for schedule(static)
    for (int64_t n = 0; n < N; ++n) {
      for (int j = 0; j < r; ++j) { rho[j] = Z[n * r + j]; Zhat[n * r + j] = 0.0; }
      for (int l = 0; l < L; ++l) {
        const double* Cl = C + (int64_t)l * K * r;
        double best = INFINITY, second = INFINITY;
        int32_t kbest = 0;
        for (int k = 0; k < K; ++k) {
          double D = 0.0;
          for (int j = 0; j < r; ++j) { double t = rho[j] - Cl[(int64_t)k * r + j]; D += t * t; }
          if (D < best) { second = best; best = D; kbest = k; }   /* strict <: lowest index wins ties */
          else if (D < second) second = D;
        }
        if (forced && forced[n * L + l] >= 0) kbest = forced[n * L + l];
        codes[n * L + l] = kbest;
        if (d1) d1[n * L + l] = best;
        if (d2) d2[n * L + l] = second;
        for (int j = 0; j < r; ++j) {
          double c = Cl[(int64_t)kbest * r + j];
          rho[j] -= c;
          Zhat[n * r + j] += c;
        }
      }
      if (rho_out) for (int j = 0; j < r; ++j) rho_out[n * r + j] = rho[j];
    }
    free(rho);
  }
}

/* squared distance of one residual to one codeword (used by tests of the near-tie rule) */
double mapl_oracle_sqdist(int r, const double* rho, const double* c) {
  double D = 0.0;
  for (int j = 0; j < r; ++j) { double t = rho[j] - c[j]; D += t * t; }
  return D;
}

/* dequantise: Zhat = sum_l C[l,codes_l,:]  (receiver side of P:149) */
void mapl_oracle_dequant(int64_t N, int r, int L, int K, const int32_t* codes, const double* C,
                         double* Zhat) {
#pragma omp parallel for schedule(static)
  for (int64_t n = 0; n < N; ++n) {
    for (int j = 0; j < r; ++j) Zhat[n * r + j] = 0.0;
    for (int l = 0; l < L; ++l)
      for (int j = 0; j < r; ++j)
        Zhat[n * r + j] += C[((int64_t)l * K + codes[n * L + l]) * r + j];
  }
}

/* ---------------------------------------------------------------- reconstruction (Eq. 2, Eq. 3)
 * Hhat = Zhat U^T + A[tok] B.   ra == 0 or A == NULL: no anchor.                          */
void mapl_oracle_decode(int64_t N, int d, int r, int ra, const double* Zhat, const double* U,
                        const int32_t* tok, const double* A, const double* B, double* Hhat) {
#pragma omp parallel for schedule(static)
  for (int64_t n = 0; n < N; ++n) {
    for (int i = 0; i < d; ++i) {                 /* (Zhat U^T)[n,i] */
      double s = 0.0;
      for (int j = 0; j < r; ++j) s += Zhat[n * r + j] * U[(int64_t)i * r + j];
      Hhat[n * d + i] = s;
    }
    if (A && ra > 0)                              /* + (A[tok_n,:] B)[i] */
      for (int q = 0; q < ra; ++q) {
        double a = A[(int64_t)tok[n] * ra + q];
        for (int i = 0; i < d; ++i) Hhat[n * d + i] += a * B[(int64_t)q * d + i];
      }
  }
}

/* ---------------------------------------------------------------- backward (Alg. 1 l.4)
 * Given g = dL/dHhat, with L a function of Hhat = Zhat U^T + A[tok] B, Zhat = Z + sg(Zhat - Z)
 * (straight-through, reading S7), Z = H U:
 *   gz = g U                         (what crosses the wire backwards)
 *   dU = g^T Zhat + H^T gz           (decode-side + encode-side term, reading S8; H NULL -> first only)
 *   dH = gz U^T
 *   dA[v,:] = sum_{n: tok_n = v} g[n,:] B^T     (E_small trainable)
 *   dB = A[tok]^T g                  (P_p is frozen in the paper; computed on request)
 * Any output pointer may be NULL (skipped).  dA must have room for V*ra.                 */
void mapl_oracle_backward(int64_t N, int d, int r, int ra, int V, const double* g, const double* H,
                          const double* Zhat, const double* U, const int32_t* tok, const double* A,
                          const double* B, double* gz, double* dU, double* dA, double* dB,
                          double* dH) {
  double* gzl = gz ? gz : (double*)malloc(sizeof(double) * (size_t)N * r);
#pragma omp parallel for schedule(static)
  for (int64_t n = 0; n < N; ++n) {               /* gz[n,:] = sum_i g[n,i] U[i,:] */
    for (int j = 0; j < r; ++j) gzl[n * r + j] = 0.0;
    for (int i = 0; i < d; ++i) {
      double a = g[n * d + i];
      for (int j = 0; j < r; ++j) gzl[n * r + j] += a * U[(int64_t)i * r + j];
    }
  }
  if (dU) {
#pragma omp parallel for schedule(static)
    for (int i = 0; i < d; ++i) {                 /* dU[i,:] = sum_n g[n,i] Zhat[n,:] + sum_n H[n,i] gz[n,:] */
      for (int j = 0; j < r; ++j) dU[(int64_t)i * r + j] = 0.0;
      for (int64_t n = 0; n < N; ++n) {
        double a = g[n * d + i];
        for (int j = 0; j < r; ++j) dU[(int64_t)i * r + j] += a * Zhat[n * r + j];
      }
      if (H)
        for (int64_t n = 0; n < N; ++n) {
          double a = H[n * d + i];
          for (int j = 0; j < r; ++j) dU[(int64_t)i * r + j] += a * gzl[n * r + j];
        }
    }
  }
  if (dH) {
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < N; ++n)
      for (int i = 0; i < d; ++i) {
        double s = 0.0;
        for (int j = 0; j < r; ++j) s += gzl[n * r + j] * U[(int64_t)i * r + j];
        dH[n * d + i] = s;
      }
  }
  if (dA && ra > 0) {
    double* gA = (double*)malloc(sizeof(double) * (size_t)N * ra);
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < N; ++n)               /* gA[n,q] = sum_i g[n,i] B[q,i] */
      for (int q = 0; q < ra; ++q) {
        double s = 0.0;
        for (int i = 0; i < d; ++i) s += g[n * d + i] * B[(int64_t)q * d + i];
        gA[n * ra + q] = s;
      }
    for (int64_t q = 0; q < (int64_t)V * ra; ++q) dA[q] = 0.0;
    for (int64_t n = 0; n < N; ++n)               /* serial scatter: duplicates add in token order */
      for (int q = 0; q < ra; ++q) dA[(int64_t)tok[n] * ra + q] += gA[n * ra + q];
    free(gA);
  }
  if (dB && ra > 0) {
#pragma omp parallel for schedule(static)
    for (int q = 0; q < ra; ++q) {                /* dB[q,:] = sum_n A[tok_n,q] g[n,:] */
      for (int i = 0; i < d; ++i) dB[(int64_t)q * d + i] = 0.0;
      for (int64_t n = 0; n < N; ++n) {
        double a = A[(int64_t)tok[n] * ra + q];
        for (int i = 0; i < d; ++i) dB[(int64_t)q * d + i] += a * g[n * d + i];
      }
    }
  }
  if (!gz) free(gzl);
}

/* ---------------------------------------------------------------- tangent projection (Eq. 4)
 * xi = G - U sym(U^T G),  sym(M) = (M + M^T)/2.                                 */
void mapl_oracle_tangent(int d, int r, const double* U, const double* G, double* xi) {
  double* S = (double*)calloc((size_t)r * r, sizeof(double));
#pragma omp parallel for schedule(static)
  for (int a = 0; a < r; ++a)                     /* S[a,:] = sum_i U[i,a] G[i,:] */
    for (int i = 0; i < d; ++i) {
      double u = U[(int64_t)i * r + a];
      for (int b = 0; b < r; ++b) S[a * r + b] += u * G[(int64_t)i * r + b];
    }
#pragma omp parallel for schedule(static)
  for (int i = 0; i < d; ++i) {                   /* xi[i,:] = G[i,:] - sum_a U[i,a] sym(S)[a,:] */
    for (int b = 0; b < r; ++b) xi[(int64_t)i * r + b] = G[(int64_t)i * r + b];
    for (int a = 0; a < r; ++a) {
      double u = U[(int64_t)i * r + a];
      for (int b = 0; b < r; ++b) xi[(int64_t)i * r + b] -= u * 0.5 * (S[a * r + b] + S[b * r + a]);
    }
  }
  free(S);
}

/* ---------------------------------------------------------------- retraction by thin QR
 * Q of the Householder QR of Y [d,r] (d >= r, full column rank), signs fixed so that
 * diag(R) > 0 -- the unique factor (north_star "a retraction, either QR ...", reading S17).
 * R (upper triangular [r,r]) is written when non-NULL.                                   */
void mapl_oracle_qr(int d, int r, const double* Y, double* Q, double* R) {
  double* W = (double*)malloc(sizeof(double) * (size_t)d * r);   /* working copy -> R on top */
  double* V = (double*)calloc((size_t)d * r, sizeof(double));    /* Householder vectors */
  double* beta = (double*)malloc(sizeof(double) * (size_t)r);
  double* sv = (double*)malloc(sizeof(double) * (size_t)r);
  memcpy(W, Y, sizeof(double) * (size_t)d * r);
  for (int k = 0; k < r; ++k) {
    double nrm = 0.0;
    for (int i = k; i < d; ++i) nrm += W[(int64_t)i * r + k] * W[(int64_t)i * r + k];
    nrm = sqrt(nrm);
    double x0 = W[(int64_t)k * r + k];
    double alpha = (x0 >= 0.0) ? -nrm : nrm;              /* avoid cancellation */
    double vnorm2 = 0.0;
    for (int i = k; i < d; ++i) {
      double v = W[(int64_t)i * r + k] - (i == k ? alpha : 0.0);
      V[(int64_t)i * r + k] = v;
      vnorm2 += v * v;
    }
    beta[k] = (vnorm2 > 0.0) ? 2.0 / vnorm2 : 0.0;
    for (int j = k; j < r; ++j) sv[j] = 0.0;               /* W <- (I - beta v v^T) W */
    for (int i = k; i < d; ++i) {
      double v = V[(int64_t)i * r + k];
      for (int j = k; j < r; ++j) sv[j] += v * W[(int64_t)i * r + j];
    }
    for (int i = k; i < d; ++i) {
      double v = beta[k] * V[(int64_t)i * r + k];
      for (int j = k; j < r; ++j) W[(int64_t)i * r + j] -= v * sv[j];
    }
  }
  /* Q = H_0 H_1 ... H_{r-1} [I_r; 0] */
  for (int i = 0; i < d; ++i)
    for (int j = 0; j < r; ++j) Q[(int64_t)i * r + j] = (i == j) ? 1.0 : 0.0;
  for (int k = r - 1; k >= 0; --k) {
    for (int j = 0; j < r; ++j) sv[j] = 0.0;
    for (int i = k; i < d; ++i) {
      double v = V[(int64_t)i * r + k];
      for (int j = 0; j < r; ++j) sv[j] += v * Q[(int64_t)i * r + j];
    }
    for (int i = k; i < d; ++i) {
      double v = beta[k] * V[(int64_t)i * r + k];
      for (int j = 0; j < r; ++j) Q[(int64_t)i * r + j] -= v * sv[j];
    }
  }
  /* sign fix: diag(R) > 0 */
  for (int k = 0; k < r; ++k) {
    double sgn = (W[(int64_t)k * r + k] < 0.0) ? -1.0 : 1.0;
    for (int i = 0; i < d; ++i) Q[(int64_t)i * r + k] *= sgn;
    if (R) for (int j = 0; j < r; ++j) R[k * r + j] = (j >= k) ? sgn * W[(int64_t)k * r + j] : 0.0;
  }
  free(W); free(V); free(beta); free(sv);
}

/* ---------------------------------------------------------------- retraction by Newton-Schulz
 * X_0 = Y; X_{j+1} = X_j (3I - X_j^T X_j)/2, `iters` times (north_star: "a fixed number of
 * Newton-Schulz polar iterations, with the count stated" -- 5, configs[4]; reading S11: the
 * classical cubic iteration, no pre-scaling; needs sigma_max(Y) < sqrt(3)).              */
void mapl_oracle_newton_schulz(int d, int r, int iters, const double* Y, double* X) {
  double* M = (double*)malloc(sizeof(double) * (size_t)r * r);
  double* T = (double*)malloc(sizeof(double) * (size_t)d * r);
  memcpy(X, Y, sizeof(double) * (size_t)d * r);
  for (int it = 0; it < iters; ++it) {
#pragma omp parallel for schedule(static)
    for (int a = 0; a < r; ++a) {                 /* M[a,:] = (3I - X^T X)[a,:] / 2 */
      for (int b = 0; b < r; ++b) M[a * r + b] = 0.0;
      for (int i = 0; i < d; ++i) {
        double x = X[(int64_t)i * r + a];
        for (int b = 0; b < r; ++b) M[a * r + b] += x * X[(int64_t)i * r + b];
      }
      for (int b = 0; b < r; ++b) M[a * r + b] = 0.5 * ((a == b ? 3.0 : 0.0) - M[a * r + b]);
    }
#pragma omp parallel for schedule(static)
    for (int i = 0; i < d; ++i) {                 /* T[i,:] = sum_a X[i,a] M[a,:] */
      for (int b = 0; b < r; ++b) T[(int64_t)i * r + b] = 0.0;
      for (int a = 0; a < r; ++a) {
        double x = X[(int64_t)i * r + a];
        for (int b = 0; b < r; ++b) T[(int64_t)i * r + b] += x * M[a * r + b];
      }
    }
    memcpy(X, T, sizeof(double) * (size_t)d * r);
  }
  free(M); free(T);
}

/* ---------------------------------------------------------------- Stiefel step
 * xi = tangent(U,G); Y = U - lr xi; U+ = qf(Y) (retraction 0) or NS_iters(Y) (retraction 1).
 * (Eq. 4 + P:124 Eq. 7 with the retraction north_star names.)  xi_out may be NULL. */
void mapl_oracle_stiefel_step(int d, int r, const double* U, const double* G, double lr,
                              int retraction, int ns_iters, double* U_out, double* xi_out) {
  double* xi = (double*)malloc(sizeof(double) * (size_t)d * r);
  double* Y = (double*)malloc(sizeof(double) * (size_t)d * r);
  mapl_oracle_tangent(d, r, U, G, xi);
  for (int64_t q = 0; q < (int64_t)d * r; ++q) Y[q] = U[q] - lr * xi[q];
  if (retraction == 0) mapl_oracle_qr(d, r, Y, U_out, NULL);
  else mapl_oracle_newton_schulz(d, r, ns_iters, Y, U_out);
  if (xi_out) memcpy(xi_out, xi, sizeof(double) * (size_t)d * r);
  free(xi); free(Y);
}

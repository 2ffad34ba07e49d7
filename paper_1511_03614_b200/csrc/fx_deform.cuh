// fx_deform.cuh -- contour deformation of the physical region (formula DESIGN.md
// R11) at one point, shared by the interpreter kernels (fx_kernels_cplx.cu) and the native kernels
// (fx_jit_template_cplx.cu), so that both tiers do the same arithmetic in the same order:
//     g_k  = dF/dx_k (x), H_kl = d2F/dx_k dx_l (x)         from the sector's real gradient/Hessian program
//     z_k  = x_k - i*lambda*x_k*(1-x_k)*g_k
//     J_kl = delta_kl (1 - i*lambda*(1-2x_k) g_k) - i*lambda*x_k(1-x_k) H_kl
//     det J                                                complex N x N elimination in registers (R12)
#ifndef FX_DEFORM_CUH
#define FX_DEFORM_CUH

#include "fx_math.cuh"

// slot of H_kl (k <= l) in the gradient/Hessian program's outputs: the gradient first, then the upper
// triangle row by row
template <int N>
__device__ __forceinline__ constexpr int fx_hess_slot(int k, int l) {
  return N + k * N - k * (k - 1) / 2 + (l - k);
}

// det J without pivoting, on half the matrix.  With s_k = x_k(1-x_k) > 0 and L = diag(lambda s_k),
//     J = D - i L H,  D = diag(1 - i lambda (1-2x_k) g_k),  H real symmetric
// is similar to the complex SYMMETRIC matrix  L^-1/2 J L^1/2 = I - i S,
//     S_kl = delta_kl lambda (1-2x_k) g_k + lambda sqrt(s_k s_l) H_kl      (real symmetric),
// so det J = det(I - i S).  I - i S has the positive definite real part I: every leading minor is
// prod_j (1 - i mu_j) with real mu_j (|minor| >= 1), elimination without pivoting cannot break down
// and is stable (growth factor < 3 for symmetric B + iC with B positive definite, Higham, Accuracy
// and Stability of Numerical Algorithms, sect. 10.4), and only the lower triangle is carried:
// N(N+1)/2 complex entries in registers instead of N^2, half the multiply-adds, no row exchanges.
// DESIGN.md R12 ("any elimination order is correct up to rounding").
template <int N>
__device__ __forceinline__ cplx fx_det_sym(cplx (&A)[N][N] /* lower triangle l <= r used */) {
  cplx det{1.0, 0.0};
#pragma unroll
  for (int c = 0; c < N; ++c) {
    const cplx piv = A[c][c];
    det = t_mul(det, piv);
    if (c + 1 < N) {
      const cplx inv = t_rdivc(1.0, piv);
#pragma unroll
      for (int r = c + 1; r < N; ++r) {
        const cplx mn = t_neg(t_mul(A[r][c], inv));
#pragma unroll
        for (int l = c + 1; l <= r; ++l) A[r][l] = t_fma(mn, A[l][c], A[r][l]);  // A[c][l] = A[l][c]
      }
    }
  }
  return det;
}

// gh(slot): the gradient (slots 0..N-1) and upper Hessian values of F at the point.
// Returns det J and fills zi[k] = Im z_k (Re z_k = x_k).
template <int N, class GH>
__device__ __forceinline__ cplx fx_jacobian_det(double lambda, const double (&xv)[N], const double (&xbv)[N], GH gh,
                                                double (&zi)[N]) {
  cplx A[N][N];
  double rs[N];  // sqrt(lambda x_k (1-x_k))
#pragma unroll
  for (int k = 0; k < N; ++k) {
    const double xk = xv[k], xb = xbv[k], gk = gh(k);
    const double ls = lambda * (xk * xb);
    zi[k] = -(ls * gk);
    rs[k] = sqrt(ls);
    A[k][k] = cplx{1.0, -fma(ls, gh(fx_hess_slot<N>(k, k)), lambda * (xb - xk) * gk)};  // 1 - 2x = xbar - x
#pragma unroll
    for (int l = 0; l < k; ++l) A[k][l] = cplx{0.0, -((rs[k] * rs[l]) * gh(fx_hess_slot<N>(l, k)))};
  }
  return fx_det_sym<N>(A);
}

#endif

// plan_host.hpp — plan-time host code of the CUDA library (steps 1.1–1.3).
// Independent of oracle/: different base eigen-solver (implicit-shift QL on the tridiagonal; Householder
// reduction first for the dense cyclic operator of a periodic direction),
// own operator assembly and own refinement code.
#pragma once

#include <vector>

namespace tpt {

struct Operator1D {
    int n = 0;
    int bc = 0;
    std::vector<double> w;      // cell widths, n                     (paper's Delta x_i, D = diag(w))
    std::vector<double> delta;  // centre spacings at faces, n+1      (paper's Delta x_{i-1/2})
    std::vector<double> a, b, c;  // Eq. 4 sub/main/super diagonals with boundary rows, n each
};

// true iff n >= 2 and faces are finite and strictly increasing
bool faces_valid(int n, const double *xf);

// Eq. 3–4 with mirror-ghost boundary rows (readings A1–A3); bc: 0 Neumann,
// 1 Dirichlet, 2 periodic (cyclic corners kept in a[0], c[n-1], reading A17; needs n >= 3).
void build_operator(int n, const double *xf, int bc, Operator1D &op);

// Eigen-decomposition of T~ = D^{1/2} T D^{-1/2} (Eq. 5): lambda[n] descending (mode 0 smoothest),
// q[n*n] row-major with q[i*n+m] = component i of mode m; Neumann null pair set analytically;
// sign convention sum_i q_im sqrt(w_i) >= 0.  Returns 0 on success, <0 if QL failed to converge or
// the refined basis misses the accuracy rule (orthogonality defect > 1e-11).
// base_kind: 0 = implicit QL with the local relative deflation test (the plan's solver); 1 = the same iteration with a
// deliberately crude normwise deflation test (test only: the refinement must absorb the difference).
int eigen_decompose(const Operator1D &op, std::vector<double> &lambda, std::vector<double> &q, int base_kind = 0);

}  // namespace tpt

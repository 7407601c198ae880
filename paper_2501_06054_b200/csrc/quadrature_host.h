// Host-side quadrature tables for the CUDA tracer (DESIGN.md R-A9, R-A11).
// Independent of oracle/: nodes are eigenvalues of the Jacobi matrix found by Sturm
// bisection, weights are Christoffel numbers from the orthonormal three-term recurrence.
#pragma once
#include <vector>

namespace sas {

// Gauss rule of the symmetric tridiagonal Jacobi matrix (diag a[0..n), off-diagonal b[1..n)),
// normalised so that the weights sum to 1.
void gauss_from_jacobi(const std::vector<double>& a, const std::vector<double>& b, std::vector<double>& x,
                       std::vector<double>& w);

// Schulz distribution of unit mean and relative width p: n nodes (size multipliers) + weights.
void schulz_rule(double p, int n, std::vector<double>& s, std::vector<double>& w);

// Gaussian tilt of std sigma truncated to [-3 sigma, 3 sigma]: n Gauss-Legendre nodes + weights.
void gauss_tilt_rule(double sigma, int n, std::vector<double>& d, std::vector<double>& w);

}  // namespace sas

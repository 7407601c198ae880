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

// Gauss-Legendre rule on [0, 1]: n nodes (ascending) and weights summing to 1.
void legendre_rule_01(int n, std::vector<double>& x, std::vector<double>& w);

// Hayter-Penfold MSA (DESIGN.md R-S2): mean-spherical closure for hard spheres of unit diameter (packing eta)
// with the Yukawa repulsion beta u(x) = gam exp(-k (x - 1)) / x, x > 1, through the Baxter / Hoye-Blum
// factorisation.  out = {a, b, E, C', D'}: Q(x) = a (x^2 - 1)/2 + b (x - 1) + E exp(-k x) - C' inside the core,
// D' exp(-k (x - 1)) outside; *g_contact = g(1+) = a + b - k C'.  Newton's method on five equations, continued
// from the Percus-Yevick solution in 20 steps of gam.  Returns false if the iteration does not converge.
bool msa_solve(double eta, double gam, double k, double out[5], double* g_contact);

}  // namespace sas

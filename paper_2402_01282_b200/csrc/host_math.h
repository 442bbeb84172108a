// host_math.h -- declarations of the host-side kernel build (filters.cpp).
#pragma once
#include <vector>

namespace s2w {

int scale_count(int L, double lambda);                                  // J: smallest integer with lambda^J >= L
int scale_bandlimit(int j, int L, double lambda, bool multires);        // L_j  (Eq. 38)
int scaling_bandlimit(int L, double lambda, int J0, bool multires);     // L_s
void kappa_profiles(int L, double lambda, int J0, int J, std::vector<double> &kappa, std::vector<double> &ksc);
void zeta_tiling(int L, int N, std::vector<double> &zeta);
void gauss_laguerre2(int P, std::vector<double> &x, std::vector<double> &q);
void laguerre_basis(int Pband, const std::vector<double> &x, double tau, std::vector<double> &K);
double pi_d();

}  // namespace s2w

// Host build of paper_1702_02939_b200/csrc/avm_math.cuh (the header is plain C++ when not
// compiled by nvcc): lets the CPU test-suite check the device math against mpmath.
#include "../paper_1702_02939_b200/csrc/avm_math.cuh"

extern "C" {
void h_log_unit(long n, const double* u, double* out) { for (long i = 0; i < n; ++i) out[i] = avm::log_unit(u[i]); }
void h_cos_2pi(long n, const double* u, double* out) { for (long i = 0; i < n; ++i) out[i] = avm::cos_2pi(u[i]); }
void h_sincos_any(long n, const double* t, double* s, double* c) { for (long i = 0; i < n; ++i) avm::sincos_any(t[i], s + i, c + i); }
}

// normbp.cuh - launchers of the matrix-message (norm network) BP kernels, see normbp.cu.
#pragma once
#include "common.cuh"
#include <algorithm>

namespace pepo {

// W (4 ci x 4 co, ld 4 ci) = I_4 (x) M (ci x co, ld ldm): turns launch_site_apply into "contract one leg
// of a site tensor with a matrix" (the chi x chi absorb / de-absorb GEMM of PAPER.md:L318, L336)
int launch_kron_i4(cudaStream_t st, const double* M, int ci, int co, int ldm, double* W);
// message from the cross Gram G ((4 chi)^2): Pauli trace, symmetrise, Frobenius-normalise, damp, delta
int launch_norm_msg(cudaStream_t st, const double* G, int chi, const double* old, double damping, double* out,
                    double* raw, unsigned long long* delta_bits, int* flag);
int launch_frob_dot(cudaStream_t st, const double* A, const double* B, int n, double* out);
int launch_psqrt_build(cudaStream_t st, const double* U, const double* V, const double* s, int chi, double eps,
                       double* S, double* Sinv);
// M = diag(v) (mode 0), diag(sqrt v) (1), diag(1/sqrt v) (2)
int launch_set_diag(cudaStream_t st, const double* v, int chi, int mode, double* M);

}  // namespace pepo

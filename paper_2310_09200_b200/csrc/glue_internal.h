// Shared by glue.cu and eig_subspace.cu only: library handles of the glue workspace and the leading-eigenpair solver.
#pragma once
#include "internal.h"

#include <cublas_v2.h>
#include <cusolverDn.h>

cublasHandle_t bb_glue_blas(GlueWork* g);
cusolverDnHandle_t bb_glue_solver(GlueWork* g);
cusolverDnParams_t bb_glue_params(GlueWork* g);
SubspaceWork** bb_glue_subspace_slot(GlueWork* g);

// Leading m eigenpairs of nb Hermitian matrices C (n x n complex128, contiguous, both triangles valid) by block
// subspace iteration (eig_subspace.cu). *used = 1: the fast path produced the result — *n_vec >= m Ritz vectors
// (n x *n_vec, ascending eigenvalue order, *stride_v elements between matrices) and values (*stride_l between matrices);
// *used = 0: not applicable or not converged — C is untouched and the caller runs the full eigensolve.
int bb_subspace_top_eigs(GlueWork* g, cudaStream_t st, int nb, int n, int m, cuDoubleComplex* C, const cuDoubleComplex** vecs,
                         int64_t* stride_v, const double** lams, int64_t* stride_l, int* n_vec, int* used, int* launches);

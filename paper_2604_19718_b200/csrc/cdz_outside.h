// cdz_outside.h -- workspace of the outside (adjoint) pass, shared by cdz_outside.cu (cell kernel) and cdz_usage.cu (finishing kernels).
#pragma once
#include <string.h>

#include "cdz_internal.h"

constexpr int ORING = 36;  // diagonals kept of the per-cell ring tables: a closing pair lies at most 32 diagonals above its inner pair
constexpr int XU = 27;     // interior totals u = l1 + l2 = 4..30 with l1, l2 >= 2
constexpr int SLEN = 31;   // loop-side stretches have 0..30 positions
constexpr int XRING = 6;   // diagonals kept of the adjoint X_u recursions (PART 1 of a diagonal may run while PART 0 is 4 diagonals ahead)
constexpr int SRING = 4;   // diagonals kept of the PART 0 -> PART 1 scratch records

__host__ __device__ inline int scr_size(int MS, int ML, int MR, int nps) {
  return (2 * ML * MR + 16 * MS * MS + 8 * MS * MS + MS * MS + nps * MS * MS + 1 + 1) & ~1;
}

// roles of an operator (one accumulator each: a single writer per launch, summed in this order at the end)
enum { ROLE_PL = 0, ROLE_PR, ROLE_CL, ROLE_CR, ROLE_IL, ROLE_IR, ROLE_B1L, ROLE_B1R, ROLE_E, ROLE_ML, ROLE_M1, ROLE_EXT, NROLE };
// roles of a short unpaired stretch E(s, s+len-1)
enum { AES_XL = 0, AES_XR, AES_Z1R, AES_Z2L, AES_BL, AES_BR, AES_NROLE };

struct Adj {
  double *AM2, *AM2T;  // S x S   M2-bar, row (i,a) column (j+1,c); and transposed
  double *AML;         // S x S   Qml-bar
  double *AM1T;        // S x S   Qm1-bar transposed: row (j+1,c), column (i,a)
  double *AET;         // S x S   E-bar transposed: row (e+1,c), column (s,a) = adjoint of E(s,e)[a,c]
  double *QM1, *QMT;   // S x S   plain transposes of QM1T / QM (contiguous operands of the two split-point gathers)
  double *AB;          // LS x RS Qb-bar
  double *AX, *AXB;    // Qext-bar: [(n+1)][MS] and over the bond index space
  double *IB;          // [ORING][n][16 MS^2]  I(i,j)[slot][a'][c']
  double *IBS;         // [ORING][n][MS^2]     I summed over the slots (bulges of size >= 2 and the multiloop closure do not see the pair type)
  double *RD;          // [ORING][n][ML MR + MS^2 + ML MS + MR MS]  adjoints of DD | GI | D1 | D2T of the cell, pushed by its closing cells
  double *XA, *XB;     // [XRING][n][27 MS^2]  adjoint row / column recursions of the interior-loop bodies
  double *SC;          // [SRING][n][scr_size]  per-cell scratch records handed from PART 0 to PART 1 of the cell kernel
  double *AES;         // [AES_NROLE][n][SLEN][MS^2]  adjoints of the loop-side stretches, by role, start position and length
  double *U;           // [NROLE][nops] operator usages by role
  int* status;         // [0] = 1 when a marginal left [0,1] or a sum rule failed (cdz_marginals_status)
  int ML, MR;
  size_t nops;
};

size_t cdz_outside_carve(const cdz_tt* tt, void* base, Adj* out);
int cdz_launch_outside(cdz_tables* t, const Adj& A, size_t ws_bytes, double* bpp_dev, double* base_dev, double* codon_dev, cudaStream_t st);
int cdz_launch_usage(cdz_tables* t, const Adj& A, double* bpp_dev, double* base_dev, double* codon_dev, cudaStream_t st);

// panel.cuh -- the panel factorisation of the blocked LU (panel.cu): constants shared with the workspace layout in lu.cu.
#pragma once
#include "lu.cuh"

namespace hp {

constexpr int PANEL_NT = 256;
constexpr int PANEL_MINROWS = 128;
// exchange buffer of the register-resident panel kernel (layout: see "panel kernel, v2" below), in 8-byte words
constexpr int LL_SLOT_WORDS = 2;            // { epoch16 | 48 payload bits } x 2 = |candidate| (64 bits) + row (32 bits)
constexpr int LL_ROW_WORDS = IB * 4;        // room for IB double2 elements
constexpr size_t LL_SLOTS = 2 * (size_t)MAXG * MAXG * LL_SLOT_WORDS;     // words: one mailbox of MAXG slots per CTA and parity
constexpr size_t LL_ROWS = 2 * (size_t)(MAXG + 1) * LL_ROW_WORDS;        // words; row index MAXG = "row j"
constexpr size_t LL_WORDS = LL_SLOTS + LL_ROWS;

// Factor the m x w panel Asub (w <= IB columns, partial pivoting) with one cooperative launch: pivots to
// ipiv[c0 ..] (1-based, absolute rows c0 + .), first zero pivot to info_dev, multipliers scaled in place, the inverses of the
// w x w unit-lower / upper triangles to dl / du and the net row permutation of the batch to perm.
template <class V>
int panel_launch(cudaStream_t st, V Asub, int m, int w, int c0, int *ipiv, int *info_dev, LuWork<V> &wk, V dl, V du, int *perm);

// Block panel of a factorisation with verified diagonal pivots (toplu.cu): factors the TW-wide (w <= TW) column block at
// (c0,c0) of the n x n matrix A without interchanges -- top block in one CTA, L21 = A21 U11^-1 by one GEMM -- and counts
// refuted multipliers (|l|_1 > 1/2, zero pivots) in *wk.refuted.  dl / du receive the inverses of the top block's triangles.
template <class V> int block_panel(cudaStream_t st, int n, V A, int c0, int w, int *ipiv, int *info_dev, LuWork<V> &wk, V dl, V du);

}  // namespace hp

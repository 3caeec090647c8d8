// Term engine: builds the operator terms of PAPER.md Eq. (6) by brute-force enumeration of the
// elementary strings of PAPER.md Eq. (1), names the per-part factors, pre-sums them into
// complementary operators, and emits contraction items for the planner.
#pragma once
#include "model.h"

namespace dmrg {

struct EOp { bool cre; int orb; int spin; };   // spin 0 = up, 1 = down

// One absorbed site: new block = old block (+) site (left) or site (+) old block (right).
// Builds the new block's operator classes on the device ("renormalization steps").
std::unique_ptr<BlockSide> renormalize_block(dmrg_ctx* ctx, const BlockSide& old, int site /*1-based*/,
                                             cudaStream_t st, double* flops_out);

// Vacuum block left of site 1 / right of site L.
std::unique_ptr<BlockSide> vacuum_block(dmrg_ctx* ctx, bool is_left, cudaStream_t st);

// Frees the pre-summed (complementary) classes a two-site problem attached to a block; the carried ones stay.
void drop_presummed(BlockSide& b, bool su2);

// Two-site problem at bond (k, k+1): psi layout, complementary operators, apply plan, diagonal.
void prepare_superblock(dmrg_ctx* ctx, cudaStream_t st);

// SU(2)-adapted counterparts (engine_su2.inc; sector labels (N, 2S), reduced matrix elements).
std::unique_ptr<BlockSide> renormalize_block_su2(dmrg_ctx* ctx, const BlockSide& old, int site, cudaStream_t st,
                                                 double* flops_out);
namespace su2e { std::unique_ptr<BlockSide> vacuum_block_su2(dmrg_ctx* ctx, bool is_left, cudaStream_t st); }
void prepare_superblock_su2(dmrg_ctx* ctx, cudaStream_t st);

}  // namespace dmrg

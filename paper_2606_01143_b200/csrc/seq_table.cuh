// seq_table.cuh -- the sequences of one launch, packed back to back along the token axis
// (a suffix wave of Phase B, or the single prefix sequence of Phase A / C).  Passed by value as a
// kernel parameter; holds no arithmetic of the method.
#pragma once

namespace pf {

constexpr int kMaxSeqs = 32;  // sequences per launch (the host splits longer waves)

struct SeqTable {
    int n;
    int cu[kMaxSeqs + 1];   // token offset of sequence s in the packed tensors
    int pqs[kMaxSeqs + 1];  // prefix sums of ceil(Ls / 64): first global 64-row query sub-tile of s
    int ckt[kMaxSeqs + 1];  // prefix sums of ceil(Ls / 128): first global 128-row tile of s
};

// Visible part of the prefix source: up to kMaxRanges row ranges of the K1/V1 buffer (the whole
// prefix [0, Lp) by default; the ancestors of a node for tree-structured data).
constexpr int kMaxRanges = 8;

struct PrefixRanges {
    int n;
    int start[kMaxRanges];      // first row of range r
    int len[kMaxRanges];        // rows of range r
    int tile0[kMaxRanges + 1];  // prefix sums of ceil(len / 128): first 128-row tile of range r
    // tile index -> (range, first row of the tile in the buffer, valid rows of the tile)
    __host__ __device__ void locate(int tile, int& row0, int& valid) const {
        int r = 0;
        while (r + 1 < n && tile0[r + 1] <= tile) ++r;
        const int i = tile - tile0[r];
        row0 = start[r] + i * 128;
        valid = len[r] - i * 128;
    }
};

}  // namespace pf

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

}  // namespace pf

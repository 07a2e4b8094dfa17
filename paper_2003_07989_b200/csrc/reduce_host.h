// reduce_host.h -- the serial remainder of the reduction of the non-apparent columns (Algorithm 2,
// PAPER.md:182-200; "submatrix reduction") after the device has reduced every
// column against the apparent ones (reduce.cu).  NOT the hot path: it runs on the host, as the whole
// submatrix reduction does in the paper, and is timed and reported separately.
#pragma once
#include <stdint.h>
#include <vector>

struct HostReduceIn {
    int n, d;
    const uint32_t* K;        // host copy of the key matrix (lower triangle)
    const uint64_t* binom;    // host binomial table, k-major, stride n+1
    int bstride;
    uint32_t thr_key;         // cofacets with key < thr_key are above the threshold
    uint32_t n_keys;          // number of distinct keys (keys are 0 .. n_keys-1)
    const uint64_t* cols;     // packed column records of the non-apparent columns, coboundary order
    int64_t ncols;
    int cbits;
    int tbits;                // bits of the row index field
    const uint64_t* pre;      // per column, from the device pre-reduction against the apparent columns: 0 = zero column,
                              // ~0 = not pre-reduced, else (key << tbits | cidx(t)) + 1 with t not an apparent row; may be NULL
};

struct HostReduceOut {
    std::vector<uint64_t> piv_t, piv_s; // pivots found, in processing order
    std::vector<uint32_t> piv_key_t, piv_key_s;
    std::vector<uint64_t> ess_s;        // zero columns
    std::vector<uint32_t> ess_key;
    std::vector<int64_t> piv_col, ess_col; // position of the column in `cols`
    int64_t additions = 0;
    int64_t lookups = 0;
};

void host_reduce_columns(const HostReduceIn& in, HostReduceOut& out);

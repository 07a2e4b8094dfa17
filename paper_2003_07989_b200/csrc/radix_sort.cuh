// radix_sort.cuh -- interface of the hand-written onesweep radix sort (no CUB, no Thrust).
// Step a6 / a9 of DESIGN.md: the paper's "GPU-sort" (pair array sorted by
// row).
#pragma once
#include "common.cuh"

#define RIPS_SORT_MAX_PASSES 8
#define RIPS_SORT_MAX_BINS 256

struct SortPlan {
    int npasses;
    int shift[RIPS_SORT_MAX_PASSES];
    int bits[RIPS_SORT_MAX_PASSES];
    i64 tile_items;
};

// Digits covering bits [lo_bit, hi_bit): 8-bit digits from lo_bit up, the last one narrower (digit r = byte r of the field).
SortPlan sort_make_plan(int lo_bit, int hi_bit);

// Scratch the sort needs besides the ping-pong buffer, in bytes (status words, histograms, ticket).
size_t sort_scratch_bytes(i64 n, const SortPlan& plan);

struct SortTimes {
    cudaEvent_t ev[3]; // optional: [0] before histogram, [1] after histogram, [2] after the last pass
    bool enabled;
    bool external = false; // the stream is being captured: record the events as external event nodes
};

// Stable LSD sort of n u64 records by the plan's digits, ascending.  `a` holds the input, `b` is the
// ping-pong buffer; returns (via *result) which of the two holds the sorted data (a if the number
// of passes is even).  scratch: sort_scratch_bytes(n, plan) device bytes.  launches += kernels run.
// hist_ready: the caller zeroed the scratch head with sort_prepare_fused and a producer kernel has
// already accumulated the raw digit counts of every pass into sort_hist_ptr(scratch)[pass][256]
// (FusedHist in kernels.cuh); the sort then skips its own histogram read of the records.
// ballot_passes: bit p set = the 32 records of a warp mostly differ in the digit of pass p (keys of edges, mantissa bits):
// that pass ranks by ballots instead of MATCH (radix_sort.cu, onesweep_pass_kernel).  Any value gives the same result.
// n_dev (optional): the number of records lives on the device (u64); n is then its upper bound (launch size, scratch size)
// and the kernels sort min(*n_dev, n) records.  Whatever the count, the sorted data ends in *result.
cudaError_t sort_u64(u64* a, u64* b, i64 n, const SortPlan& plan, void* scratch, cudaStream_t stream,
                     u64** result, SortTimes* times, i64* launches, bool hist_ready = false,
                     u32 ballot_passes = 0, const u64* n_dev = nullptr);
// (clears the whole scratch of a sort of n records: histograms, tickets, the status words of every pass)
cudaError_t sort_prepare_fused(void* scratch, i64 n, const SortPlan& plan, cudaStream_t stream);

// The sort's scratch as a static device array (radix_sort.cu): its device address on the CURRENT device and its size.
// No allocation; the address is asked for once per device.  Shared by every caller: see the note at the array.
#define RIPS_SORT_STATIC_BYTES (16u << 20)
#define RIPS_SORT_STATIC_MAX_RECORDS (1ll << 22)
#define RIPS_SORT_STATIC_MAX_DEVICES 64
cudaError_t sort_static_scratch(void** ptr, size_t* bytes);
u64* sort_hist_ptr(void* scratch);

// Internal declarations shared by the host planner (tangram_host.cpp) and the CUDA side
// (tangram_decode.cu).  Not part of the C ABI.
#ifndef TANGRAM_INTERNAL_H_
#define TANGRAM_INTERNAL_H_

#include <stdint.h>

namespace tangram {

// Records the thread-local error string and returns `code`.
int fail(int code, const char* fmt, ...);

// Item as the kernels read it (32 bytes, 16-byte aligned).  Same fields as tangram_item except that
// `cluster` is replaced by the CSR offset of the (request, cluster) page-table row, so the kernel
// reaches a page id with one load: tbl_pages[tbl_row + token / P].
struct alignas(16) DeviceItem {
    int32_t req, kv_head, tbl_row, slot, tok_begin, tok_end, part_slot, n_parts;
};
static_assert(sizeof(DeviceItem) == 32, "DeviceItem must be 32 bytes");

}  // namespace tangram

// Debug build (python -m paper_2606_06302_b200.build --spin-limit N -> libtangram_spin.so): every device loop that
// spins on a flag ANOTHER CTA (or another grid) sets -- the query-staging flags, the per-sequence part counters of the
// in-grid merge, the per-row ready flags of the compaction gather -- gives up after N polls: it prints which wait it
// was and where, and traps, so a deadlock ends as a CUDA error of the launch instead of a kernel that never returns.
// N = 0 (the shipped library): the checks compile to nothing.
#ifndef TANGRAM_SPIN_LIMIT
#define TANGRAM_SPIN_LIMIT 0
#endif
#define TANGRAM_WAIT_Q_FLAG 1      // producer warp: the item's query block has not been staged (tangram_decode_attention_host)
#define TANGRAM_WAIT_SEQ_PARTS 2   // tail phase: a sequence's parts of this launch have not all been published
#define TANGRAM_WAIT_ROW_READY 3   // compaction gather: the select kernel has not published the row's indices
#if defined(__CUDACC__) && TANGRAM_SPIN_LIMIT > 0
#include <cstdio>
#define TANGRAM_SPIN_INIT unsigned long long tangram_spins_ = 0
#define TANGRAM_SPIN_POLL(which, what)                                                                              \
    do {                                                                                                            \
        if (++tangram_spins_ > static_cast<unsigned long long>(TANGRAM_SPIN_LIMIT)) {                               \
            printf("tangram: spin limit %llu hit in wait %d (index %d), block %d thread %d\n",                      \
                   static_cast<unsigned long long>(TANGRAM_SPIN_LIMIT), which, static_cast<int>(what),              \
                   static_cast<int>(blockIdx.x), static_cast<int>(threadIdx.x));                                    \
            __trap();                                                                                               \
        }                                                                                                           \
    } while (0)
#else
#define TANGRAM_SPIN_INIT (void)0
#define TANGRAM_SPIN_POLL(which, what) (void)0
#endif

#endif

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

#endif

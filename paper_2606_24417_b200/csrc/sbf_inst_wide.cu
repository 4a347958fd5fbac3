// sbf_inst_wide.cu — specialised streaming instances for DNA k-mers wider than one 64-bit word (33 <= k <= 64; P:153,
// P:435, readings A20/A21): the same thread-serial kernels with a 5- or 6-word register window and m-mers / s-mers of
// more than 32 symbols folded to 64 bits before hashing.  The sliding minimum covers k-m+1 <= 39 and the sliding OR
// k-s <= 16; every other (k, m, s, H) with k > 32 runs wide_tile_kernel.  See sbf_dispatch.h.
#include "sbf_dispatch.h"
#ifndef SBF_ONLY_DEFAULT // tuning builds compile the default instance only
namespace sbfk {
static const KernelEntry kTable[] = {
    SBF_ENTRY(63, 31, 60, 4),
    SBF_ENTRY(63, 40, 60, 4),
    SBF_ENTRY(51, 25, 48, 4),
    SBF_ENTRY(51, 31, 48, 4),
    SBF_ENTRY(47, 24, 44, 4),
    SBF_ENTRY(33, 16, 30, 4),
    SBF_ENTRY(64, 41, 64, 8),
};
static const TableRegistration kReg(kTable, (int)(sizeof(kTable) / sizeof(kTable[0])));
} // namespace sbfk
#endif

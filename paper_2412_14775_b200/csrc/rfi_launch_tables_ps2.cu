// rfi_launch_tables_ps2.cu -- per-sample-mask instantiations 128..191 of the tables kernel (rfi_tables_ps.inc).
#define RFI_PS_PART 2
#include "rfi_tables_ps.inc"

namespace rfi_host {
int launch_tables_ps_part2(int idx, const rfi::KParams& kp, cudaStream_t st) {
    static constexpr auto table = make_table(std::make_integer_sequence<int, 64>{});
    return table[idx](kp, st);
}
}  // namespace rfi_host

// rfi_launch_tables_ps0.cu -- per-sample-mask instantiations 0..63 of the tables kernel (rfi_tables_ps.inc).
#define RFI_PS_PART 0
#include "rfi_tables_ps.inc"

namespace rfi_host {
int launch_tables_ps_part0(int idx, const rfi::KParams& kp, cudaStream_t st) {
    static constexpr auto table = make_table(std::make_integer_sequence<int, 64>{});
    return table[idx](kp, st);
}
}  // namespace rfi_host

// rfi_launch_batched_mask_f32.cu -- fp32-storage instantiations of rfi_batched_mask_kernel.
#define RFI_BM_FP16 0
#include "rfi_launch_batched_mask.inc"

// rfi_launch_batched_mask_f16.cu -- fp16-storage instantiations of rfi_batched_mask_kernel.
#define RFI_BM_FP16 1
#include "rfi_launch_batched_mask.inc"

// gsp_stage1.cu — tiled stage-1 kernel (channel -> subband shift-and-sum): placeholder
// translation unit until the shared-memory kernel lands; the generic stage 1 lives in
// gsp_kernels.cu.
#include "gsp_internal.h"

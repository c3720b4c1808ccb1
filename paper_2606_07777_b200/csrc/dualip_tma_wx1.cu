// dualip_tma_wx1.cu -- every k_grad_tma instantiation that writes x (WX = true): evaluations whose caller asked for x
// (dualip_grad with x, the final evaluation of dualip_solve with x_out, every DUALIP_RED_CSC evaluation).
#include "dualip_grad_tma.cuh"

const void* dualip_tma_kernel_wx1(int G, int M, bool acc_smem, bool gbox) {
    return dualip_dev::TmaKernelTable<true>::get(G, M, acc_smem, gbox);
}

// dualip_tma_wx0.cu -- every k_grad_tma instantiation that never writes x (WX = false): the kernels dualip_solve's
// iteration loop and x-less dualip_grad calls launch.  A translation unit of its own so that it compiles in parallel
// with dualip_tma_wx1.cu and dualip_api.cu (paper_2606_07777_b200/build.py).
#include "dualip_grad_tma.cuh"

const void* dualip_tma_kernel_wx0(int G, int M, bool acc_smem, bool gbox) {
    return dualip_dev::TmaKernelTable<false>::get(G, M, acc_smem, gbox);
}

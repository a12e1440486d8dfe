// panel_f32.cu -- fp32 instantiations of the register-resident cooperative panel kernel.
#include "panel.cuh"

namespace ctqr {

template <int IB, int RPT>
static cudaError_t launch(PanelArgs<float>& pa, int G, cudaStream_t st) {
    void* args[] = {(void*)&pa};
    return cudaLaunchCooperativeKernel((void*)panel_geqr2_kernel<float, IB, RPT, kPanelThreads>, dim3(G),
                                       dim3(kPanelThreads), args, 0, st);
}

cudaError_t panel_launch_f32(int ib, int rpt, PanelArgs<float>& pa, int G, cudaStream_t st) {
    if (ib == 16 && rpt == 1) return launch<16, 1>(pa, G, st);
    if (ib == 16 && rpt == 2) return launch<16, 2>(pa, G, st);
    if (ib == 16 && rpt == 4) return launch<16, 4>(pa, G, st);
    if (ib == 16 && rpt == 8) return launch<16, 8>(pa, G, st);
    if (ib == 8 && rpt == 2) return launch<8, 2>(pa, G, st);
    if (ib == 8 && rpt == 8) return launch<8, 8>(pa, G, st);
    if (ib == 32 && rpt == 1) return launch<32, 1>(pa, G, st);
    if (ib == 32 && rpt == 2) return launch<32, 2>(pa, G, st);
    if (ib == 32 && rpt == 4) return launch<32, 4>(pa, G, st);
    return cudaErrorInvalidValue;
}

}  // namespace ctqr

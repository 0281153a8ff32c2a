// sgw_pass_inst.cu -- compiled once per supported axis length (-DSGW_N=<N>): instantiates every
// fused pass kernel for that length and exports one launcher, sgw_pass_launch_<N>.
#include "sgw_ops.cuh"

#ifndef SGW_N
#error "compile with -DSGW_N=<axis length>"
#endif

namespace sgw {

template <int MODE, class Op>
static int launch(const PassCall* c) {
    constexpr int N = SGW_N;
    Op op;
    op.p = c->p;
    const int threads = c->gm.B * pass_threads_per_pencil<N>();
    const size_t smem = (size_t)c->gm.B * pass_smem_per_pencil<N>();
    if (threads > 256) return -1;
    auto kern = pass_kernel<N, MODE, Op>;
    if (smem > 48 * 1024) {
        static bool attr_done = false;
        if (!attr_done) {
            if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024) != cudaSuccess)
                return -4;
            attr_done = true;
        }
    }
    kern<<<(unsigned)c->ntiles, threads, smem, c->stream>>>(c->gm, c->in, c->tw, op);
    return cudaGetLastError() == cudaSuccess ? 0 : -4;
}

}  // namespace sgw

#define SGW_CAT_(a, b) a##b
#define SGW_CAT(a, b) SGW_CAT_(a, b)

extern "C" int SGW_CAT(sgw_pass_launch_, SGW_N)(const sgw::PassCall* c) {
    using namespace sgw;
    switch (c->kind) {
        case K_RT_STORE: return launch<MODE_RT, OpStore>(c);
        case K_RT_ACC: return launch<MODE_RT, OpAcc>(c);
        case K_RT_HFIN: return launch<MODE_RT, OpHFin>(c);
        case K_RT_CHEB: return launch<MODE_RT, OpCheb>(c);
        case K_RT_TD: return launch<MODE_RT, OpTD>(c);
        case K_RT_MUL3D: return launch<MODE_RT, OpMul3D>(c);
        case K_FWD: return launch<MODE_FWD, OpStore>(c);
        case K_INV: return launch<MODE_INV, OpStore>(c);
        default: return -1;
    }
}

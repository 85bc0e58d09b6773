// fft_zt_inst.cu -- instantiates the (z,t) pass of the tiled FFT (fft_zt.cuh) for ONE Nz, given on the
// command line as -DLGF_ZT_NA=<Nz>, and every Nt in {8, 12, 16, 24, 32, 48, 64}, FP64 and FP32.
// build.py compiles this file once per Nz; fft_tiled.cu dispatches on Nz to the functions defined here.
#include "fft_zt.cuh"

#ifndef LGF_ZT_NA
#error "compile with -DLGF_ZT_NA=<Nz>"
#endif
#define LGF_CAT2(a, b) a##b
#define LGF_CAT(a, b) LGF_CAT2(a, b)
#define LGF_ZT_FN(name) LGF_CAT(name, LGF_ZT_NA)

namespace lgf {

#define LGF_NT_SWITCH(EXPR_D, EXPR_F)                            \
    switch (nt) {                                                \
    case 8: { constexpr int NB = 8; return prec == 0 ? (EXPR_D) : (EXPR_F); }   \
    case 12: { constexpr int NB = 12; return prec == 0 ? (EXPR_D) : (EXPR_F); } \
    case 16: { constexpr int NB = 16; return prec == 0 ? (EXPR_D) : (EXPR_F); } \
    case 24: { constexpr int NB = 24; return prec == 0 ? (EXPR_D) : (EXPR_F); } \
    case 32: { constexpr int NB = 32; return prec == 0 ? (EXPR_D) : (EXPR_F); } \
    case 48: { constexpr int NB = 48; return prec == 0 ? (EXPR_D) : (EXPR_F); } \
    case 64: { constexpr int NB = 64; return prec == 0 ? (EXPR_D) : (EXPR_F); } \
    default: break;                                              \
    }

// x-columns per tile for (Nz, Nt) = (LGF_ZT_NA, nt), 0 if the pair is not instantiated
int LGF_ZT_FN(zt_columns_na)(int nt, int prec)
{
    LGF_NT_SWITCH((ZTC<double, LGF_ZT_NA, NB>::C), (ZTC<float, LGF_ZT_NA, NB>::C))
    return 0;
}
// kernel attributes (shared-memory opt-in); 0 on success
int LGF_ZT_FN(zt_setup_na)(int nt, int prec)
{
    LGF_NT_SWITCH((setup_zt_n<double, LGF_ZT_NA, NB>()), (setup_zt_n<float, LGF_ZT_NA, NB>()))
    return 1;
}
int LGF_ZT_FN(zt_launch_na)(const FftArgs &a, cudaStream_t st)
{
    const int nt = a.geo.N[3], prec = a.prec;
    LGF_NT_SWITCH((launch_zt_n<double, LGF_ZT_NA, NB>(a, st)), (launch_zt_n<float, LGF_ZT_NA, NB>(a, st)))
    return 1;
}
// the two-launch form (LGF_OPT_FFT_PASSES = 4): is it instantiated for this pair, and its launcher
int LGF_ZT_FN(zt_has_half_na)(int nt)
{
    const int prec = 0;
    LGF_NT_SWITCH((zt_pipe_pair(LGF_ZT_NA, NB) ? 1 : 0), 0)
    return 0;
}
int LGF_ZT_FN(zt_launch_half_na)(const FftArgs &a, int inverse, cudaStream_t st)
{
    const int nt = a.geo.N[3], prec = a.prec;
    LGF_NT_SWITCH((launch_zt_half_n<double, LGF_ZT_NA, NB>(a, inverse, st)), (launch_zt_half_n<float, LGF_ZT_NA, NB>(a, inverse, st)))
    return 1;
}

} // namespace lgf

// k_amp_direct.cu -- instantiations of the direct amplitude kernels (k_amplitude.cuh, NB = 0): one phasor per pair,
// by MUFU (NPOLY = 0) or by polynomial on the FMA and ALU pipes (NPOLY = QT: the accurate variant).  Moving only one
// or two of a thread's eight phasors to the FMA pipe was measured SLOWER than all-MUFU on B200 (C3: 1820 -> 1448 /
// 1351 Gpair/s): the polynomial phasor costs ~26 issue cycles against 6 + 16 XU cycles (profiles/r2_*.md).
// 16 points per thread at 2 blocks per SM, which lifted the recurrence kernels, does not help here: the kernel is bound by
// the XU pipe, not by per-line work (C3, per-particle split: 0.652 -> 0.564; with 2 / 3 / 4 of the 16 phasors by polynomial
// 0.464 / 0.382 / 0.385).
#include "k_amplitude.cuh"

namespace nms {

template <int MODE, int QT, int NCH, int NPOLY>
static amp_kernel_t pick(bool split)
{
    if constexpr (NCH == 4) { if (split) return (amp_kernel_t)k_amp<MODE, QT, true, 4, 0, 4, NPOLY, 0>; }
    return (amp_kernel_t)k_amp<MODE, QT, false, 4, 0, NCH, NPOLY, 0>;
}

template <int MODE>
static amp_kernel_t pick_mode(int qt, bool split, int nch, int npoly)
{
    if (nch == 1 && split) return nullptr;           // a one-channel object split runs the four-channel kernel
    if constexpr (MODE != 2) if (qt == 8) {
        if (nch == 1) return npoly == 0 ? pick<MODE, 8, 1, 0>(false) : npoly == 8 ? pick<MODE, 8, 1, 8>(false) : nullptr;
        return npoly == 0 ? pick<MODE, 8, 4, 0>(split) : npoly == 8 ? pick<MODE, 8, 4, 8>(split) : nullptr;
    }
    if (qt == 4) {
        if (nch == 1) return npoly == 0 ? pick<MODE, 4, 1, 0>(false) : npoly == 4 ? pick<MODE, 4, 1, 4>(false) : nullptr;
        return npoly == 0 ? pick<MODE, 4, 4, 0>(split) : npoly == 4 ? pick<MODE, 4, 4, 4>(split) : nullptr;
    }
    return nullptr;
}

amp_kernel_t amp_kernel_direct(int mode, int qt, bool split, int nch, int npoly, bool uni)
{
    (void)uni;   // block-uniform abscissae were measured slower in the direct kernels (C3: 0.652 -> 0.618)
    switch (mode) {
    case 0: return pick_mode<0>(qt, split, nch, npoly);
    case 1: return pick_mode<1>(qt, split, nch, npoly);
    case 2: return pick_mode<2>(qt, split, nch, npoly);
    default: return nullptr;
    }
}

}  // namespace nms

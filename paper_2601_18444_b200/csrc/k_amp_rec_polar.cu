// k_amp_rec_polar.cu -- instantiations of the line-recurrence amplitude kernels (k_amplitude.cuh, NB > 0) for
// MODE = 0 (polar detector): NB exactly evaluated points per QT, rotations or the three-term recurrence, phasors of
// the bases and of the step by MUFU or by polynomial.
#include "k_amplitude.cuh"

namespace nms {

template <int QT, int NB, int NCH, int REC3>
static amp_kernel_t pick(bool split, bool poly)
{
    if constexpr (NCH == 4) if (split)
        return poly ? (amp_kernel_t)k_amp<0, QT, true, 4, NB, 4, 1, REC3> : (amp_kernel_t)k_amp<0, QT, true, 4, NB, 4, 0, REC3>;
    return poly ? (amp_kernel_t)k_amp<0, QT, false, 4, NB, NCH, 1, REC3> : (amp_kernel_t)k_amp<0, QT, false, 4, NB, NCH, 0, REC3>;
}

amp_kernel_t amp_kernel_rec_polar(int qt, int nb, bool split, int nch, bool poly, bool rec3, bool uni, bool sh)
{
    // accurate variant with a step phase within a quarter cycle: rotations (the default of precision 2) or three-term
    if (sh && poly && qt == 8 && nb == 1 && nch == 4) {
        if (rec3) return split ? (amp_kernel_t)k_amp<0, 8, true, 4, 1, 4, 1, 1, false, true> : (amp_kernel_t)k_amp<0, 8, false, 4, 1, 4, 1, 1, false, true>;
        return split ? (amp_kernel_t)k_amp<0, 8, true, 4, 1, 4, 1, 0, false, true> : (amp_kernel_t)k_amp<0, 8, false, 4, 1, 4, 1, 0, false, true>;
    }
    // 16 points per thread at 2 blocks per SM (four channels, not split): the fast variant with 2 exact points and the
    // three-term recurrence (the arithmetic of 8 points with 1), the accurate variant with 1 exact point and rotations
    if (qt == 16) {
        if (nch == 4 && !split) {
            if (!poly && rec3 && nb == 2) return (amp_kernel_t)k_amp<0, 16, false, 2, 2, 4, 0, 1>;
            if (poly && !rec3 && nb == 1)
                return sh ? (amp_kernel_t)k_amp<0, 16, false, 2, 1, 4, 1, 0, false, true> : (amp_kernel_t)k_amp<0, 16, false, 2, 1, 4, 1, 0>;
            return nullptr;
        }
    }
    // the default fast kernel with block-uniform line abscissae (n1 a multiple of 128): C5 0.783 -> 0.804 of the roofline
    if (uni && qt == 8 && nb == 1 && nch == 4 && !poly && rec3)
        return split ? (amp_kernel_t)k_amp<0, 8, true, 4, 1, 4, 0, 1, true> : (amp_kernel_t)k_amp<0, 8, false, 4, 1, 4, 0, 1, true>;
    if (nch == 1) {
        if (split) return nullptr;
        if (qt == 16 && nb == 4) return rec3 ? pick<16, 4, 1, 1>(false, poly) : pick<16, 4, 1, 0>(false, poly);
        if (qt == 8 && nb == 2) return rec3 ? pick<8, 2, 1, 1>(false, poly) : pick<8, 2, 1, 0>(false, poly);
        return nullptr;
    }
    if (qt != 8) return nullptr;
    switch (nb) {
    case 1: return rec3 ? pick<8, 1, 4, 1>(split, poly) : pick<8, 1, 4, 0>(split, poly);
    case 2: return rec3 ? pick<8, 2, 4, 1>(split, poly) : pick<8, 2, 4, 0>(split, poly);
    case 3: return rec3 ? nullptr : pick<8, 3, 4, 0>(split, poly);
    case 4: return rec3 ? nullptr : pick<8, 4, 4, 0>(split, poly);
    default: return nullptr;
    }
}

}  // namespace nms

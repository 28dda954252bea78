// pm_slab.cuh -- z-slab decomposition of the exchange step (Eq. 3).
//
// One ctx per rank holds the planes [z0, z0 + nz) of a domain that is periodic in x and y inside the rank and cut along z.
// Particles live with their host cell (L43).  The only non-local step is Step 2 (L97): the z ghost planes of a rank's buffer
// mesh are added to the real zones of its two z neighbours.  The planes of one channel are contiguous in memory, so a slab
// is packed as [channel][g planes][ny + 2g][row pitch] -- x and y ghost cells included, UNfolded: the receiver's fold then
// adds the images of a cell in the same fixed order (z image, y image, x image) as the single-domain fold does, which is what
// Appendix A asks of the buffer sum (L623-627: contributions summed in a fixed order of the contributing grids) and what
// makes one rank talking to itself bit-identical to the periodic fold.  Stale tiles (pm_tiles.cuh) are packed as the zeros
// they stand for.
// Step 4 needs eta and v_old in the cells of the NEIGHBOUR that a boundary sink reached (L79); the paper does not say how they
// get there (R16): here the return mesh carries g ghost planes per side and the owners' boundary planes are copied into them
// after the apply pass (contiguous planes, no packing; pm_slab_desc in include/pm.h).
#pragma once
#include "pm_device.cuh"
#include "pm_tiles.cuh"

namespace pm {

// side 0: planes k in [-g, 0) (they go to the lower neighbour); side 1: planes k in [nz, nz + g) (to the upper neighbour)
template <int NCH>
__global__ void __launch_bounds__(256) k_slab_pack(const DevP P, const double *__restrict__ buf, const Tiles T,
                                                   double *__restrict__ send_lo, double *__restrict__ send_hi) {
    const long long per_side = (long long)P.g * P.pk;                 // cells of one channel of one slab
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= 2 * per_side) return;
    const int side = t >= per_side ? 1 : 0;
    const long long r = t - side * per_side;
    const int p = (int)(r / P.pk);
    const long long inplane = r - (long long)p * P.pk;
    const int jj = (int)(inplane / P.pj), ii = (int)(inplane - (long long)jj * P.pj);   // ghosted plane coordinates
    const int i = ii - P.gx, j = jj - P.g, k = side ? P.nz + p : p - P.g;
    unsigned f = 0;
    if (i >= -P.g && i < P.nx + P.g) f = T.live[tile_index(P, i, j, k)];      // (the pad columns beyond the g ghost cells hold nothing)
    const long long src = (long long)(k + P.g) * P.pk + inplane;
    double *dst = side ? send_hi : send_lo;
#pragma unroll
    for (int ch = 0; ch < NCH; ++ch) {
        const bool live = ch == 0 ? (f & kLiveK) : (ch == kChK ? (f != 0) : (f & kLiveN));
        dst[(long long)ch * per_side + r] = live ? buf[(long long)ch * P.Nb + src] : 0.0;
    }
}

}  // namespace pm

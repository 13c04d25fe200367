// fn_fixed_step.cuh -- the PAPER'S OWN range query as a comparison kernel, not part
// of the product path: "Range sensing uses fixed-step samples along each beam.  Samples from all
// environments are queried in distance blocks, and beams with a detected obstacle are removed from
// subsequent blocks"; its ablation baseline evaluates all samples of all rays
// (PAPER.md:192, :199).  Here: one thread per beam, sample k at distance k * delta from the sensor
// origin (first sample at 0, reading G5), occupancy of the cell containing the sample from the packed
// map (outside = occupied), range = distance of the first occupied sample, none below r_max => r_max.
// kBlockwise: the march stops after the block of 32 samples in which it first hit ("removed from
// subsequent blocks"); otherwise every sample up to r_max is evaluated ("All samples").  fp32 sample
// positions, like the tensor operations it stands for.  Both variants return the same ranges.
#pragma once
#include "fn_common.cuh"

namespace fn {

struct FixedStepArgs {
    MapDev map;
    const BeamPose* poses;       // sensing poses (cos/sin of the heading; origin via ouM of both orientations)
    const double2* beam_cs;      // [B]
    int n, B;
    float delta_cells;           // sample spacing in cells
    int n_samples;               // ceil(r_max / delta)
    float rmax, rho;
    float* out_ranges;           // [n][B]
};

template <bool kBlockwise>
__global__ void __launch_bounds__(256) fixed_step_kernel(FixedStepArgs a) {
    const unsigned idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (unsigned)a.n * (unsigned)a.B) return;
    const unsigned e = idx / (unsigned)a.B, j = idx - e * (unsigned)a.B;
    const BeamPose* p = a.poses + e;
    const double2 cs = a.beam_cs[j];
    const float dx = (float)(p->c * cs.x - p->s * cs.y), dy = (float)(p->s * cs.x + p->c * cs.y);
    const float ox = (float)(p->o[0].ouM - (kMagic + (double)kCellShift));
    const float oy = (float)(p->o[1].ouM - (kMagic + (double)kCellShift));
    int first = a.n_samples;                                       // index of the first occupied sample
    for (int k0 = 0; k0 < a.n_samples; k0 += 32) {
        for (int k = k0; k < min(k0 + 32, a.n_samples); ++k) {
            const float t = (float)k * a.delta_cells;
            const int cj = __float2int_rd(fmaf(t, dx, ox)), ci = __float2int_rd(fmaf(t, dy, oy));
            if (occ_global(a.map, ci, cj)) first = min(first, k);
        }
        if (kBlockwise && first < a.n_samples) break;
    }
    const float r = (float)first * a.delta_cells * a.rho;
    a.out_ranges[idx] = first < a.n_samples ? fminf(r, a.rmax) : a.rmax;
}

}  // namespace fn

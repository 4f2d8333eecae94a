// gw_accounting.cu — executed-flop and launch bookkeeping reported through gw_executed_flops / gw_launch_count.
#include "gw_common.cuh"

// stage 2: the two transforms as executed (complex tile MMAs, 2048 flops each) plus the nominal count of the
// Cholesky solve (potrf + two triangular solves with naux right-hand sides, 8*(7/6) n^3 ... = 28/3 n^3 flops).
static double stage2_flops(const gw_problem *p) {
  GwDims d = gw_dims(p);
  const double len = (double)d.nq * d.naux * d.naux;
  const double nblocks = (len + 63) / 64;
  const double tr = nblocks * 8.0 * (((d.nw + 7) / 8) * ((d.ntau + 3) / 4) + ((d.ntau + 7) / 8) * ((d.nw + 3) / 4)) * 2048.0;
  const double sol = (double)d.nw * d.nq * (28.0 / 3.0) * d.naux * (double)d.naux * d.naux;
  return tr + sol;
}

void gw_stage_flops(const gw_problem *p, double *o) {
  o[0] = gw_stage1_flops(p); o[1] = stage2_flops(p); o[2] = gw_stage3_flops(p); o[3] = gw_stage4_flops(p);
}

// kernels launched by the four hot calls: stage 1: 1; stage 2: set_info + transform + dyson + transform; stage 3: 1;
// stage 4: exchange + reduce  (the three 256-byte cudaMemsetAsync of the work counters are not kernels)
int gw_stage_launches(const gw_problem *p) { (void)p; return 1 + 4 + 1 + 2; }

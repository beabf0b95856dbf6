/* Prints sizeof / offsetof of every struct of include/fdtd_llg.h as the C compiler lays them out.
 * tests/test_abi_cpu.py compiles this (gcc, plain C: the header must be a C header) and compares
 * the numbers with the ctypes mirrors in paper_2103_12819_b200/binding.py. */
#include <stddef.h>
#include <stdio.h>

#include "fdtd_llg.h"

#define S(T) printf("sizeof " #T " %zu\n", sizeof(T))
#define F(T, f) printf("offsetof " #T " " #f " %zu\n", offsetof(T, f))

int main(void) {
  S(fdtd_llg_options);
  F(fdtd_llg_options, bc); F(fdtd_llg_options, enable_llg); F(fdtd_llg_options, h_bias);
  F(fdtd_llg_options, ani_hk); F(fdtd_llg_options, ani_axis); F(fdtd_llg_options, llg_tol);
  F(fdtd_llg_options, llg_max_iter); F(fdtd_llg_options, use_graph);
  F(fdtd_llg_options, scalar_material_mask); F(fdtd_llg_options, kernel_path);
  F(fdtd_llg_options, time_scheme); F(fdtd_llg_options, pml); F(fdtd_llg_options, pml_r0);
  F(fdtd_llg_options, pml_order); F(fdtd_llg_options, merge_h); F(fdtd_llg_options, slab_ext);
  S(fdtd_llg_stats);
  F(fdtd_llg_stats, steps); F(fdtd_llg_stats, time); F(fdtd_llg_stats, iters_last);
  F(fdtd_llg_stats, iters_max); F(fdtd_llg_stats, iters_total);
  F(fdtd_llg_stats, nonconverged_halfsteps); F(fdtd_llg_stats, resid_last);
  F(fdtd_llg_stats, halfsteps); F(fdtd_llg_stats, courant); F(fdtd_llg_stats, kernel_launches);
  F(fdtd_llg_stats, magnetic_cells); F(fdtd_llg_stats, launches_per_step);
  F(fdtd_llg_stats, sweep_cells); F(fdtd_llg_stats, material_array_mask);
  F(fdtd_llg_stats, staged_sweeps); F(fdtd_llg_stats, merged_h); F(fdtd_llg_stats, staged_maxwell);
  S(fdtd_llg_slab_info);
  F(fdtd_llg_slab_info, fields_offset); F(fdtd_llg_slab_info, array_stride);
  F(fdtd_llg_slab_info, nx); F(fdtd_llg_slab_info, ny); F(fdtd_llg_slab_info, nz);
  F(fdtd_llg_slab_info, n_arrays); F(fdtd_llg_slab_info, merged_h);
  printf("enum SUB %d %d %d %d %d %d\n", FDTD_LLG_SUB_BEGIN, FDTD_LLG_SUB_HM1, FDTD_LLG_SUB_HM1_END,
         FDTD_LLG_SUB_E, FDTD_LLG_SUB_HM2, FDTD_LLG_SUB_HM2_END);
  printf("enum K_NCLASS %d\n", FDTD_LLG_K_NCLASS);
  return 0;
}

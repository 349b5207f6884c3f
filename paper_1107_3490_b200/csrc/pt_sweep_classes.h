// The classes the composed-CTA kernels are instantiated for, one list per translation unit (pt_sweep_comp<u>.cu), so
// that the units compile in parallel; pt_sweep.cu sees all of them.
//   PT_COMP(NC)       k_sweep_comp<Real, NC, ceil(NC/2), ceil(NC/4)>: 8 NC slots per chain, N in 8 NC - 7 .. 8 NC
//   PT_SEVEN(N8, N10) k_sweep_seven<Real, N8, N10>: exact fit only, for chain lengths where the 10-lane warps pay
// Every N in 17..128 has a PT_COMP class.
#pragma once
#define PT_COMP_CLASSES_0 PT_SEVEN(13, 10) PT_COMP(13)            /* N = 97..100: the throughput batch */
#define PT_COMP_CLASSES_1 PT_COMP(7) PT_COMP(8) PT_SEVEN(7, 6)    /* N = 49..64; the paper's N = 55 */
#define PT_COMP_CLASSES_2 PT_COMP(3) PT_COMP(4) PT_COMP(5)
#define PT_COMP_CLASSES_3 PT_COMP(6) PT_COMP(9)
#define PT_COMP_CLASSES_4 PT_COMP(10) PT_COMP(11)
#define PT_COMP_CLASSES_5 PT_COMP(12) PT_SEVEN(10, 8)             /* N = 80 */
#define PT_COMP_CLASSES_6 PT_COMP(14) PT_COMP(15)
#define PT_COMP_CLASSES_7 PT_COMP(16)
#define PT_COMP_UNITS 8

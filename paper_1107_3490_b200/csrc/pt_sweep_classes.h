// The (N8, N10, N16, N32) classes k_sweep_comp is instantiated for: partner-loop iterations of warps with 8, 10,
// 16 and 32 lanes per chain (L x NI slots >= N).  One list per translation unit (pt_sweep_comp<u>.cu), so that
// the units compile in parallel; pt_sweep.cu sees all of them.  Exact classes for the chain lengths of
// BASELINE.json and of the timing tables (N = 30, 55, 64, 80, 100, 128), padded classes in between:
// every N in 17..128 is covered.  PT_SEVEN(N8, N10) = k_sweep_seven, the composition "7 chains on every
// sub-partition" with the kinds of the warps fixed at compile time (class (N8, N10, -1, -1)).
#pragma once
#define PT_COMP_CLASSES_0 PT_COMP(13, 10, 7, 4) PT_SEVEN(13, 10)           /* N = 97..100; 7 chains on every sub-partition */
#define PT_COMP_CLASSES_1 PT_COMP(7, 6, 4, 2) PT_COMP(8, 7, 4, 2)          /* N = 49..56, 57..64    */
#define PT_COMP_CLASSES_2 PT_COMP(4, 3, 2, 1) PT_COMP(4, 4, 2, 1) PT_COMP(13, 11, 7, 4)   /* N = 25..30, 31..32, 101..104 */
#define PT_COMP_CLASSES_3 PT_COMP(10, 8, 5, 3) PT_COMP(9, 8, 5, 3)         /* N = 73..80, 65..72    */
#define PT_COMP_CLASSES_4 PT_COMP(16, 13, 8, 4) PT_COMP(15, 12, 8, 4)      /* N = 121..128, 113..120 */
#define PT_COMP_CLASSES_5 PT_COMP(3, 3, 2, 1) PT_COMP(5, 4, 3, 2) PT_SEVEN(7, 6)          /* N = 17..24, 33..40; N = 51..56, 7 chains on every sub-partition */
#define PT_COMP_CLASSES_6 PT_COMP(6, 5, 3, 2) PT_COMP(11, 9, 6, 3)         /* N = 41..48, 81..88    */
#define PT_COMP_CLASSES_7 PT_COMP(12, 10, 6, 3) PT_COMP(14, 12, 7, 4)      /* N = 89..96, 105..112  */
#define PT_COMP_UNITS 8

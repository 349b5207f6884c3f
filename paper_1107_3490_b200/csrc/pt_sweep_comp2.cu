// k_sweep_comp instantiations, unit 2 of pt_sweep_classes.h (one unit per file: they compile in parallel).
#include "pt_sweep_classes.h"
#define PT_COMP_UNIT 2
#define PT_COMP_CLASSES PT_COMP_CLASSES_2
#include "pt_sweep_comp.inl"

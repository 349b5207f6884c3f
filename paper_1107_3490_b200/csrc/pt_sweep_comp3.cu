// k_sweep_comp instantiations, unit 3 of pt_sweep_classes.h (one unit per file: they compile in parallel).
#include "pt_sweep_classes.h"
#define PT_COMP_UNIT 3
#define PT_COMP_CLASSES PT_COMP_CLASSES_3
#include "pt_sweep_comp.inl"

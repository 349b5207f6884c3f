// k_sweep_comp instantiations, unit 0 of pt_sweep_classes.h (one unit per file: they compile in parallel).
#include "pt_sweep_classes.h"
#define PT_COMP_UNIT 0
#define PT_COMP_CLASSES PT_COMP_CLASSES_0
#include "pt_sweep_comp.inl"

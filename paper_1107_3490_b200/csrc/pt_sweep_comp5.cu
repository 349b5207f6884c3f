// k_sweep_comp instantiations, unit 5 of pt_sweep_classes.h (one unit per file: they compile in parallel).
#include "pt_sweep_classes.h"
#define PT_COMP_UNIT 5
#define PT_COMP_CLASSES PT_COMP_CLASSES_5
#include "pt_sweep_comp.inl"

// k_sweep_comp instantiations, unit 4 of pt_sweep_classes.h (one unit per file: they compile in parallel).
#include "pt_sweep_classes.h"
#define PT_COMP_UNIT 4
#define PT_COMP_CLASSES PT_COMP_CLASSES_4
#include "pt_sweep_comp.inl"

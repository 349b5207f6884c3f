// k_sweep_comp instantiations, unit 7 of pt_sweep_classes.h (one unit per file: they compile in parallel).
#include "pt_sweep_classes.h"
#define PT_COMP_UNIT 7
#define PT_COMP_CLASSES PT_COMP_CLASSES_7
#include "pt_sweep_comp.inl"

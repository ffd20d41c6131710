// knobs.h -- private: tuning knobs of the kernels.  In the product build a knob IS its default (a constant the compiler
// folds); the library reads nothing from the environment.  Only a build with -DTBPM_EXPERIMENT (the sweeps that chose
// the defaults; tbpm_version() then ends in "+exp") exports tbpm_set_knob(name, value) and looks the knobs up at run time.
#pragma once

namespace tbpm_detail {
#ifdef TBPM_EXPERIMENT
int knob(const char *name, int dflt);
#else
inline int knob(const char *, int dflt) { return dflt; }
#endif
}  // namespace tbpm_detail

// The flux sweeps of the MHD path in the default arithmetic flavour: ak_mhd.cu compiled a second time, with AKM_FAST_TU defined
// and WITHOUT -fmad=false (build.py), so that the compiler may contract multiply-adds in PLM / PPM / WENOZ / HLLD.  See the
// comment at akm::launch_sweeps_fast in ak_mhd.cu.
#define AKM_FAST_TU 1
#include "ak_mhd.cu"

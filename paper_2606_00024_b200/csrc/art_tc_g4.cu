// art_decode_tc_kernel<G = 4, MODE, MT>: instantiations and launcher (see art_launch.h)
#define ART_TC_G 4
#include "art_tc_inst.inc"

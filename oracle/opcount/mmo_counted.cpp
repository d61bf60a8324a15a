// mmo_counted.cpp -- the oracle's own source files compiled with `double` replaced by the
// operation-counting type of opcount.hpp.  Nothing of the oracle is re-typed here: the two .c
// files are included verbatim.  Built by count_flops.py into libmmo_counted.so.
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <cmath>
#include "opcount.hpp"

#undef isfinite
#define isfinite(x) mmo_isfinite(x)
#define double cnt
#include "../mmo.h"
#include "../mmo_moments.c"
#include "../mmo_scheme.c"
#undef double
#undef isfinite

extern "C" long long mmo_opcount_get(void) { return cnt::ops; }
extern "C" void mmo_opcount_reset(void) { cnt::ops = 0; }

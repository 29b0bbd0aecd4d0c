// cp_error.cpp -- thread-local error message shared by the scheduler and the CUDA side.
#include <cstdarg>
#include <cstdio>

#include "cp.h"

static thread_local char g_cp_err[512] = "";

void cp_set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_cp_err, sizeof g_cp_err, fmt, ap);
    va_end(ap);
}

extern "C" const char* cp_last_error(void) { return g_cp_err; }

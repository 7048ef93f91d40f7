// api.cu -- error reporting and version of libmg.
#include <cstdarg>
#include <cstdio>

#include "mg_common.cuh"

static thread_local char g_err[512] = "";

void mg_set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}

extern "C" const char* mg_last_error_string(void) { return g_err; }
extern "C" int mg_version(void) { return 100; }

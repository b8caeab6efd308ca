// Thread-local last-error message behind fmx_last_error().
#include <cstdarg>
#include <cstdio>

#include "fmx.h"
#include "common.h"

static thread_local char g_err[512] = "";

int fmx_fail(int code, const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}

void fmx_clear_error() { g_err[0] = 0; }

extern "C" const char *fmx_last_error(void) { return g_err; }
extern "C" const char *fmx_version(void) { return "fmx 0.1 (sm_100a)"; }

// Shared host-side declarations of libfmx (error reporting).
#pragma once
#include <stdint.h>

// Records a thread-local message (printf-style) and returns `code`.
int fmx_fail(int code, const char *fmt, ...) __attribute__((format(printf, 2, 3)));
void fmx_clear_error();

// bb_hooks.h -- the two pieces of bb_api.cu's state that other translation units of the library
// may touch: the thread-local error message behind bb_last_error(), and the launch counter behind
// bb_launch_count().  Defined at the end of bb_api.cu.
#pragma once

namespace bb {

int report_error(int code, const char *message);   // stores the message for bb_last_error(), returns code
void count_launches(unsigned n);                   // adds n to bb_launch_count()

}  // namespace bb

"""B200-native dipolar SSCN step (arxiv 1601.04640): libdbec.so + its ctypes binding."""

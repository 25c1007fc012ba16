"""B200-native dipolar SSCN step (arxiv 1601.04640): Python binding over the C-ABI library."""

"""ringx-b200: B200-native chunked attention + LSE merge (the RingX hot path, arXiv 2507.16697).

Thin Python binding over the C-ABI library `libringx.so` (see include/ringx.h).  Importing this
package does not load the library; the first call does, and fails loudly if it is missing.
"""
__version__ = "0.1.0"

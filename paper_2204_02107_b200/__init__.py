"""B200-native DNSLABIB Navier-Stokes time step (arxiv 2204.02107).

`paper_2204_02107_b200.binding` is the thin Python layer over the C ABI in
include/dnslab.h (libdnslab.so, hand-written sm_100a CUDA kernels).  Importing the
package does not load the library; the first use does, and fails loudly if it is
missing -- there is no CPU fallback.
"""
__all__ = ["binding", "cases"]

"""B200-native nonlinear E×B term of the GX Laguerre-Hermite gyrokinetic solver (arxiv 2209.06731).

``binding`` -- ctypes binding of the C-ABI (include/gx.h); ``inputs`` -- seeded synthetic inputs;
``build`` -- nvcc build of csrc/ into libgx.so.  Nothing is imported eagerly.
"""

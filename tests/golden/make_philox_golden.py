"""Writes tests/golden/philox_curand.txt from the cuRAND *host* generator
(CURAND_RNG_PSEUDO_PHILOX4_32_10, a library routine; runs without a GPU).

cuRAND's host stream for seed s is, in groups of four 32-bit words, group e (= offset/4 + q)
= Philox4x32-10(counter = (h_lo, h_hi, e & 0xFFFF, 0), key = (s_lo, s_hi)) with h = e >> 16
(65536 interleaved subsequences), so each line is a known answer for one (key, counter) pair.  The oracle's block function
(R1) is pinned against these lines in tests/test_oracle_pins.py.
Line format: seed offset_groups q w0 w1 w2 w3 (hex); e = offset_groups + q.
"""
import ctypes as C
import os

lib = C.CDLL("libcurand.so.10")
out = []
for seed, off in [(0, 0), (1, 0), (0x123456789, 0), (0xDEADBEEFCAFEF00D, 7), (42, 0x1_0000_FFFD), (2**64 - 1, 2**40 + 3), (7, (0xABCD1234567 << 16) + 0xFFFE)]:
    g = C.c_void_p()
    assert lib.curandCreateGeneratorHost(C.byref(g), 161) == 0          # CURAND_RNG_PSEUDO_PHILOX4_32_10
    assert lib.curandSetPseudoRandomGeneratorSeed(g, C.c_ulonglong(seed)) == 0
    assert lib.curandSetGeneratorOffset(g, C.c_ulonglong(4 * off)) == 0
    buf = (C.c_uint32 * 24)()
    assert lib.curandGenerate(g, buf, C.c_size_t(24)) == 0
    for q in range(6):
        out.append("%x %x %x %08x %08x %08x %08x" % (seed, off, q, *buf[4 * q:4 * q + 4]))
    lib.curandDestroyGenerator(g)
with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "philox_curand.txt"), "w") as f:
    f.write("# cuRAND host Philox4x32-10 known answers; written by make_philox_golden.py\n")
    f.write("\n".join(out) + "\n")

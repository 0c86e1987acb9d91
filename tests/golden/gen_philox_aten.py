"""Writes tests/golden/philox_aten.txt: Philox4x32-10 blocks produced by RUNNING the host-side
engine shipped in torch's headers (ATen/core/PhiloxRNGEngine.h, class at::Philox4_32) -- an
independent third-party implementation, not the oracle and not the CUDA path.  Random123's own
kat_vectors file is not available offline, so this engine is the known-answer
source for pin P1.  Convention: key = (seed lo, seed hi); counter = (offset lo, offset hi,
subsequence lo, subsequence hi); offset counts 128-bit blocks.

Run:  python tests/golden/gen_philox_aten.py        (needs g++ and torch's headers; no GPU)
"""
import os
import subprocess
import tempfile

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
INC = os.path.join(os.path.dirname(torch.__file__), "include")

SRC = r"""
#include <ATen/core/PhiloxRNGEngine.h>
#include <cstdio>
#include <cstdint>
int main() {
  const uint64_t M = 0xFFFFFFFFFFFFFFFFull;
  const uint64_t cases[][3] = {   // seed, subsequence, offset
    {0,0,0},{1,0,0},{1,5,7},{M,M,M},{1,0,1},{1,1,0},{2,0,0},{0x123456789ABCDEFull,0xFEDCBA987654321ull,0x0F1E2D3C4B5A6978ull},
    {1,4095,999},{1,(1ull<<60)|77,0},{1,(2ull<<60)|12345,3},{7,5233139,99999},{1ull<<32,1ull<<32,1ull<<32},
    {0xDEADBEEFull,0xFFFFFFFFull,0xFFFFFFFFull},{42,0x100000000ull,0x100000000ull},{1,123456789012ull,4999}};
  for (auto& c : cases) {
    at::Philox4_32 e(c[0], c[1], c[2]);
    uint32_t r0 = e(), r1 = e(), r2 = e(), r3 = e();
    std::printf("%016llx %016llx %016llx %08x %08x %08x %08x\n", (unsigned long long)c[0],
                (unsigned long long)c[1], (unsigned long long)c[2], r0, r1, r2, r3);
  }
  return 0;
}
"""

def main():
    with tempfile.TemporaryDirectory() as d:
        src = os.path.join(d, "g.cpp")
        exe = os.path.join(d, "g")
        open(src, "w").write(SRC)
        subprocess.run(["g++", "-O1", "-std=c++17", "-I", INC, src, "-o", exe], check=True)
        out = subprocess.run([exe], check=True, capture_output=True, text=True).stdout
    hdr = ("# seed subsequence offset out0 out1 out2 out3 (hex) -- written by tests/golden/gen_philox_aten.py\n"
           "# source: at::Philox4_32 host engine, torch %s headers (third-party KAT stand-in, pin P1)\n" % torch.__version__)
    open(os.path.join(HERE, "philox_aten.txt"), "w").write(hdr + out)
    print(out)

if __name__ == "__main__":
    main()

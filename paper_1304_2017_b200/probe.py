"""Prints the two micro-benchmark tables behind DESIGN.md section 5.3 (needs a B200):

    python -m paper_1304_2017_b200.probe

1. scattered 32-byte sector loads (the record load of H's marching loop): SM-cycles per warp request against the
   number of active lanes and the shared memory held per block (= the L1 that is left);
2. RED.128 (the vector reduction of H^T): SM-cycles per lane against the address pattern within the warp.
"""
from . import binding as oat

SM, CLK = 148, 1.965e9


def main(device: int = 0):
    print("gather probe: SM-cycles per warp request (8 blocks x 128 threads per SM, one load in flight per warp)")
    print("smem KB/block | " + " | ".join(f"{m:>5d} lanes" for m in (4, 8, 10, 16, 32)))
    for kb in (0, 8, 12, 17, 25):
        row = []
        for m in (4, 8, 10, 16, 32):
            rate = oat.oat_measure_gather_rate_ex(device, m, kb)          # sectors/s
            row.append(SM * CLK * m / rate)
        print(f"{kb:>13d} | " + " | ".join(f"{v:>11.1f}" for v in row))
    print("RED.128 probe: SM-cycles per lane")
    names = ["every lane its own record", "32 consecutive records (16 sectors)", "one record per 128-B line",
             "lane pairs share a sector", "4 scattered lines x 8 records"]
    for p, n in enumerate(names):
        rate = oat.oat_measure_red_rate_ex(device, p)
        print(f"  {n:38s} {SM * CLK / rate:6.2f}")


if __name__ == "__main__":
    main()

"""FP64-pipe characterisation on the current GPU:  python -m paper_2404_12454_b200.probe

Prints the rates that DESIGN.md section 6 ("Roofline") quotes; needs a CUDA device.
"""
from . import gbd


def main():
    names = {0: "8 DFMA chains, 3 register sources", 1: "8 DFMA chains, constant-bank addend",
             2: "8 DFMA chains + 1 XOR + 1 ADD per 2 DFMA", 3: "1 dependent chain, 1 warp/SMSP"}
    print("| mode | what | FP64 inst/s | per SMSP-cycle at 1.965 GHz | note |")
    print("|---|---|---|---|---|")
    for mode in (0, 1, 2, 3):
        rate, lat = gbd.probe_fp64(mode, iters=8192 if mode != 3 else 20000)
        per = rate / 32 / (148 * 4) / 1.965e9
        note = f"latency {lat:.2f} cycles" if lat is not None else ""
        print(f"| {mode} | {names[mode]} | {rate:.4e} | {per:.3f} | {note} |")


if __name__ == "__main__":
    main()

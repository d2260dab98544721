"""python -m paper_1403_2136_b200.probe -- print the measured issue rates of the pipes the scan uses (B200 box only)."""
from . import binding as b


def main():
    import torch
    torch.cuda.set_device(0)
    print(f"# {torch.cuda.get_device_name(0)}; thread-instructions (mix rows: cells) per clock per SM; 1024 threads x 1 block per SM")
    for w, name in enumerate(b.PROBE_NAMES):
        print(f"{w:2d}  {name:82s} {b.mss_probe_pipe(w):8.2f}")
    rate, ms = b.mss_probe_dpx_peak(4096)
    print(f"--  whole-chip DPX 2:1 mix, wall clock: {rate / 1e12:.3f} T thread-instr/s ({ms:.3f} ms)")


if __name__ == "__main__":
    main()

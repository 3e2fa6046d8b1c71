"""Prints the roofline denominators measured on this GPU (nnp_measure_peaks, include/nnp.h) as one JSON line.

    python -m paper_2405_01491_b200.peaks [device]

SURVEY.md 8(d) asks for the TF32 tcgen05, fp32 FMA and SFU peaks to be micro-benchmarked and committed next to the
ncu reports: profiles/r01_peaks.md holds the output of this command on the round's B200.
"""
import json
import sys

from . import nnp


def main(argv):
    dev = int(argv[1]) if len(argv) > 1 else 0
    out = nnp.nnp_measure_peaks(dev)
    import torch
    out["device"] = torch.cuda.get_device_name(dev)
    out["sms"] = torch.cuda.get_device_properties(dev).multi_processor_count
    print(json.dumps(out))


if __name__ == "__main__":
    main(sys.argv)

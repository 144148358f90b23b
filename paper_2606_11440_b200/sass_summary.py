"""SASS mnemonic counts per kernel of the built library: `python -m paper_2606_11440_b200.sass_summary > profiles/r2_sass_summary.md`.

What proves the Blackwell-native paths (B200_PROFILING.md): UTC*MMA = tcgen05.mma, LDTM / STTM = tcgen05.ld / st,
UTCBAR = tcgen05.commit, UBLKCP = cp.async.bulk (TMA 1-D), SYNCS = mbarrier, HMMA = mma.sync, MUFU.TANH = tanh.approx,
VIMNMX.U16x2 = the packed u16 min / max of the service pass.
"""
import collections
import os
import re
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
WANT = ["UTCHMMA", "LDTM", "STTM", "UTCBAR", "UBLKCP", "SYNCS", "HMMA", "MUFU.TANH", "VIMNMX.U16x2", "STG.E.ENL2.256", "ACQBULK", "ATOMG", "REDG", "RED.", "total"]


def main():
    print("# SASS mnemonic counts per kernel (cuobjdump -sass of paper_2606_11440_b200/build/*.o, sm_100a)\n")
    print("Command: `python -m paper_2606_11440_b200.build && python -m paper_2606_11440_b200.sass_summary`\n")
    print("| kernel | " + " | ".join(WANT) + " |")
    print("|---|" + "---|" * len(WANT))
    for obj in sorted(os.listdir(os.path.join(HERE, "build"))):
        if not obj.endswith(".o"):
            continue
        out = subprocess.run(["cuobjdump", "-sass", os.path.join(HERE, "build", obj)], capture_output=True, text=True).stdout
        name, cnt = None, None
        rows = []
        for line in out.splitlines():
            m = re.match(r"\s*Function : (\S+)", line)
            if m:
                if name:
                    rows.append((name, cnt))
                name, cnt = m.group(1), collections.Counter()
                continue
            m = re.match(r"\s+/\*[0-9a-f]{4,6}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.x]+)", line)
            if m and name:
                op = m.group(1)
                cnt["total"] += 1
                for w in WANT[:-1]:
                    if op.startswith(w):
                        cnt[w] += 1
        if name:
            rows.append((name, cnt))
        for name, cnt in rows:
            dem = subprocess.run(["cu++filt", name], capture_output=True, text=True).stdout.strip() or name
            dem = dem.split("(im::Params")[0].split("(const")[0].split("(double")[0].split("(unsigned")[0].replace("im::", "").replace("void ", "").replace("(bool)", "")
            print(f"| `{dem}` ({obj}) | " + " | ".join(str(cnt[w]) for w in WANT) + " |")


if __name__ == "__main__":
    main()

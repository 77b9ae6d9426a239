#!/bin/bash
# usage: _work/ptxas.sh NL TEAM [extra flags]  -> per-kernel registers/spills
cd /root/repo/paper_2508_12033_b200/csrc
NL=$1; TEAM=$2; shift 2
nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -std=c++17 -Xcompiler -fPIC -DLRDMC_NL=$NL -DLRDMC_TEAM_TU=$TEAM "$@" -Xptxas -v -c -o /tmp/k_$NL$TEAM.o kernels.cu 2>&1 | python3 -c "
import sys,re
name=None
for ln in sys.stdin:
    m=re.search(r\"Compiling entry function '(\S+)'\",ln)
    if m: name=m.group(1); continue
    if 'spill' in ln: sp=ln.strip()
    if 'Used' in ln and name: print(name[:60], '|', sp, '|', ln.strip().replace('ptxas info    : ','')); name=None
"

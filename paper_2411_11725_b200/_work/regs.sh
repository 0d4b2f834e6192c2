#!/bin/bash
# usage: _work/regs.sh file.cu  -> kernel, regs, spills
cd /root/repo/paper_2411_11725_b200
nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3 -std=c++17 -Xcompiler -fPIC -Xptxas -v -c csrc/$1 -o /tmp/regs.o 2>&1 | python3 -c "
import sys,re,subprocess
name=None
for line in sys.stdin:
    m=re.search(r\"Compiling entry function '(\S+)'\",line)
    if m:
        name=subprocess.run(['c++filt',m.group(1)],capture_output=True,text=True).stdout.strip()
        name=re.sub(r'\(anonymous namespace\)::','',name); name=re.sub(r'\(.*','',name)
    m=re.search(r'(\d+) bytes spill stores',line)
    if m: sp=m.group(1)
    m=re.search(r'Used (\d+) registers',line)
    if m and name: print('%-40s regs %s spill %s'%(name[:40],m.group(1),sp)); name=None
"

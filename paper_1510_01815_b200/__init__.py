"""gbk-b200: B200-native batched chi^2 evaluation of GBKFIT-style disc-galaxy kinematic models
(Bekiaris et al., arXiv:1510.01815).  `gbk` holds the ctypes binding of the C-ABI library
(include/gbk.h); `workloads` the seeded synthetic inputs."""

// placeholder: replaced by the GPU table builder
#pragma once
#include "qed_device.cuh"
